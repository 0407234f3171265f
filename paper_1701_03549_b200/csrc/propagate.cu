// propagate.cu -- batched CA fire propagation (a3-a6): fire_simulate_batch.
//
// What is computed (PAPER.md:91 states, :97 ignition, :99/:133 synchronous update with one
// independent trial per burning neighbour = 1 - prod(1 - p_i) in law, :91/:145 a cell burns for one
// step, :100/:135 the run ends when the fire stops by itself; C-4):
//   t = 0: burning = burned = {ignition} if it is inside the lattice and burnable.
//   step t: for every burning cell b and direction d, target c = b + offset(d); if c is inside the
//   lattice, burnable and not burned at time t: one trial rnd(seed, sim, t, c, d) against T(c, d).
//   new = targets with >= 1 success; burned |= new; burning = new.
//
// Design: one persistent CTA per simulation, simulations handed out by a device
// counter (largest expected first), all CA steps inside ONE launch, no host round trip and no grid-wide
// barrier.  State per simulation = ONE bit plane, the SUSCEPTIBLE plane  sus = burnable & ~burned,
// stored as 8 x 8-cell tiles (one u64 per tile, so that the 3 x 3 window of a burning cell is one
// word for 56 % of the cells), plus a CELL-LEVEL FRONTIER LIST of the burning cells: work is
// proportional to the number of trials and idle lattice is never touched.  Thresholds are
// SOURCE-indexed: the 8 outgoing trials of a burning cell are one 32 B sector, read exactly once in
// the one step the cell burns.  A step:
//   phase 1  one lane per burning cell: its tile (and up to 3 neighbouring tiles) give the 3 x 3
//            susceptibility window, one 32 B load gives the 8 thresholds; the (target, direction,
//            threshold) triples of the warp are compacted into the trial queue in shared memory;
//   -- barrier: every read of `sus` for step t happens before any update of step t (synchronous update)
//   phase 2  one lane per trial: one Philox4x32-10 call, one compare; a success clears the target's
//            bit with atomicAnd, and the lane whose atomic saw the bit still set owns the new burning
//            cell and appends it to the next frontier (ballot / popc compaction).
//   -- barrier
// Lists live in shared memory and continue in a per-CTA global spill area; if the frontier outgrows
// even that, the simulation is handed to the rescue kernel below: a plain full-sweep, three-plane,
// pull-style restatement of the same rules with no lists at all.
#include "fire_internal.cuh"

namespace {

struct prop_params {
    const uint32_t* burnable;     // [H][Ww]
    const uint32_t* thr;          // [P][cells][8], source-indexed
    const int32_t*  ignitions;    // [S][2]
    const int32_t*  sim_param;    // [S]
    const uint64_t* seeds;        // [S]
    const int32_t*  sim_ids;      // [S] or null
    const uint32_t* order;        // [S] launch order or null
    uint64_t* tiles;              // [S][planes][Th][Tw] susceptible planes (planes = 1, or 2 for the asynchronous-warp kernel)
    uint32_t* plane_sel;          // [S] which plane holds the final state (asynchronous-warp kernel)
    uint32_t* out_burned;         // [S][H][Ww]
    uint32_t* out_steps;          // [S] or null
    unsigned long long* out_trials;  // [S] or null
    unsigned int* work_counter;   // [0] sims taken by the fast kernel, [1] sims handed to the rescue kernel, [2], [3] spare
    uint32_t* rescue_list;        // [S]
    uint32_t* spill;              // [grid][2 * (capQ - capQ_s) + 2 * (capA - capA_s)]
    int S, P, W, H, Ww, Tw, Th, num_sms;
    uint32_t max_steps;
    uint32_t capA_s, capQ_s;      // shared-memory entries: each frontier list, the trial queue
    uint32_t capA, capQ;          // total entries (shared + spill); capQ >= 8 * capA
    const uint8_t* ktime;         // [cells] burn time - 1 of the cell's fuel (fire_set_burn_time), or null
    const uint32_t* gt_planes;    // [kmax - 1][H][Ww] bit set iff the cell's burn time > j + 1 (rescue kernel), or null
    int kmax;                     // largest burn time (1 = every cell burns for one step)
    int32_t* out_time;            // [S][H][W] step at which every cell ignited (fire_set_time_output), or null
    const uint32_t* fit_ref;      // fire_set_fused_counts: reference bitmap [H][Ww], or null
    uint32_t* fit_counts;         // [S][2] = (I, N*) of Eq. 2, written by the finish kernel (rescued simulations: by the rescue kernel)
};

__device__ __forceinline__ uint32_t lanemask_lt()
{
    uint32_t m; asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m)); return m;
}

// Frontier entry: (y << 16) | x.  Trial item: (ty << 16) | (d << 13) | tx  (x, y < 8192): the frontier entry of the target
// with the direction in the three spare bits, so that neither side shifts coordinates around.
// Item of the trial "burning cell e spreads in direction d": item(e) + item_delta(d).
__device__ __forceinline__ uint32_t item_delta(int d)
{
    return (uint32_t)(fire_dy(d) * 65536 + fire_dx(d) + d * 8192);
}

// Threshold sector of a burning cell: ONE 256-bit load (LDG.E.256, sm_100) through the read-only path.  The table is
// read once per simulation, so the line need not stay in L1; L2 is asked to fetch the whole 128 B line with the miss, since
// the 3 neighbouring cells of the row are what the front reaches next.
struct thr_sector { uint4 a, b; };     // a = directions 0..3, b = directions 4..7
__device__ __forceinline__ thr_sector ldg_thr(const uint4* p)
{
    thr_sector v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::128B.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(v.a.x), "=r"(v.a.y), "=r"(v.a.z), "=r"(v.a.w), "=r"(v.b.x), "=r"(v.b.y), "=r"(v.b.z), "=r"(v.b.w) : "l"(p));
    return v;
}

// The same sector by two loads that ptxas keeps where they are written (it sinks the one above below the warp scan and the
// "no trials" exit to save registers, which puts the DRAM latency after the scan instead of under it).
__device__ __forceinline__ thr_sector ldg_thr_early(const uint4* p)
{
    thr_sector v;
    asm volatile("ld.relaxed.gpu.global.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.a.x), "=r"(v.a.y), "=r"(v.a.z), "=r"(v.a.w) : "l"(p));
    asm volatile("ld.relaxed.gpu.global.v4.u32 {%0,%1,%2,%3}, [%4+16];" : "=r"(v.b.x), "=r"(v.b.y), "=r"(v.b.z), "=r"(v.b.w) : "l"(p));
    return v;
}

__device__ __forceinline__ uint64_t ldcg_u64(const uint64_t* p) { return (uint64_t)__ldcg(reinterpret_cast<const unsigned long long*>(p)); }

constexpr uint32_t kM0 = 0xD2511F53u, kM1 = 0xCD9E8D57u;       // Philox4x32 multipliers
constexpr uint32_t kW0 = 0x9E3779B9u, kW1 = 0xBB67AE85u;       // Philox key bumps (Weyl constants)

// ------------------------------------------------------------------------------------------------
// Shared-memory access by 32-bit shared-window address (no generic-address arithmetic in the hot loops).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void sts64(uint32_t addr, uint32_t a, uint32_t b)
{
    asm volatile("st.shared.v2.u32 [%0], {%1, %2};" :: "r"(addr), "r"(a), "r"(b) : "memory");
}
__device__ __forceinline__ void sts32(uint32_t addr, uint32_t a)
{
    asm volatile("st.shared.u32 [%0], %1;" :: "r"(addr), "r"(a) : "memory");
}
__device__ __forceinline__ uint2 lds64(uint32_t addr)
{
    uint2 v; asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr) : "memory"); return v;
}
__device__ __forceinline__ uint32_t atoms_add(uint32_t addr, uint32_t v)
{
    uint32_t old; asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(old) : "r"(addr), "r"(v) : "memory"); return old;
}
__device__ __forceinline__ uint32_t lds32(uint32_t addr)
{
    uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory"); return v;
}

// Next simulation for this CTA, or 0xFFFFFFFF: batch order, or the order written by fire_order_kernel (largest expected
// fires first).  (Tried and dropped: CTAs of odd waves taking from the tail of the order, so that an SM hosts large and
// small fires side by side -- the large fires do get faster, 23.3 -> 21.5 ms, but the medium ones then start late and the
// launch gets longer, 25.6 -> 28.8 ms.)
__device__ __forceinline__ uint32_t next_simulation(const prop_params& prm)
{
    const unsigned int k = atomicAdd(prm.work_counter, 1u);
    if (k >= (unsigned int)prm.S) return 0xFFFFFFFFu;
    return prm.order ? prm.order[k] : k;
}

// ------------------------------------------------------------------------------------------------
// Per-step context of one simulation (everything the two pass functions need; all warp-invariant).
// ------------------------------------------------------------------------------------------------
struct step_ctx {
    // lattice / tables
    uint32_t W, Tw, Th;
    // susceptible planes: the base is the kernel parameter (a constant-bank operand of the address arithmetic); a plane is a
    // 32-bit tile offset from it, so no 64-bit pointer per simulation has to live in (or be rebuilt into) registers
    const uint64_t* tiles;
    uint32_t plane_r;             // tile offset of the plane this step READS
    uint32_t plane_w;             // tile offset of the plane this step UPDATES (the same plane in the two-phase kernel)
    uint32_t plane_w2;            // the same in 8 x 4-cell half tiles (2 * plane_w), kept in a register for the atomics
    const uint4* thr4;            // the threshold table (kernel parameter), 2 x uint4 per sector
    uint32_t thr_sec;             // first sector of this simulation's parameter vector (a table that fits in HBM has < 2^32 sectors)
    // lists
    uint32_t qs_addr, ac_addr, an_addr;   // shared-window addresses: trial queue, current frontier, next frontier
    uint32_t capQ_s, capA_s, capA;
    uint32_t* spill;              // per-CTA global spill areas (kernel parameter) and 32-bit word offsets into it:
    uint32_t qg_off, ac_off, an_off;   // trial queue (8 B entries), current frontier, next frontier beyond their shared-memory parts
    uint32_t cntQ, cntA_next, over;       // shared-window addresses of the queue counter, the next frontier's counter, the overflow flag
    uint32_t nA, nQ;
    uint32_t lane, lt;
    const uint8_t* ktime;         // burn-time variant only
    int32_t* time_base;           // burn-time variant only: ignition times of this simulation, or null
    uint32_t t;                   // burn-time variant only: the step being computed
};

// Appends `entry` of the lanes with `flag` to the next frontier list (shared memory, then the global spill, then overflow).
__device__ __forceinline__ void append_next(const step_ctx& c, bool flag, uint32_t entry)
{
    const uint32_t m = __ballot_sync(0xFFFFFFFFu, flag);
    if (m == 0u) return;                                           // warp-uniform
    uint32_t base = 0;
    if (c.lane == 0) base = atoms_add(c.cntA_next, (uint32_t)__popc(m));
    base = __shfl_sync(0xFFFFFFFFu, base, 0);
    if (flag) {
        const uint32_t pos = base + __popc(m & c.lt);
        if (pos < c.capA_s) sts32(c.an_addr + 4u * pos, entry);
        else if (pos < c.capA) __stcg(c.spill + (c.an_off + (pos - c.capA_s)), entry);
        else sts32(c.over, 1u);
    }
}

// Phase 1 for K units of 32 burning cells (units u0, u0 + ustride, ...; all of them exist: u * 32 < nA).
// Lanes past the end of the list re-read the last entry and contribute nothing.
// kBT (fuel-dependent burn-out time, R-21): bits 29..31 of a frontier entry = the steps the cell stays active AFTER this one;
// a cell that has some left appends itself to the next frontier (it is a source again next step).
template <int K, bool kBT = false>
__device__ __forceinline__ uint32_t cells_pass(const step_ctx& c, uint32_t u0, uint32_t ustride)
{
    uint32_t e[K], win[K];
    uint64_t tc[K], th[K], tv[K], td[K];
    uint4 Ta[K], Tb[K];
    bool live[K];
#pragma unroll
    for (int k = 0; k < K; ++k) {
        uint32_t i = (u0 + (uint32_t)k * ustride) * 32u + c.lane;
        live[k] = i < c.nA;
        i = live[k] ? i : c.nA - 1u;
        e[k] = (i < c.capA_s) ? lds32(c.ac_addr + 4u * i) : __ldcg(c.spill + (c.ac_off + (i - c.capA_s)));
        const uint32_t x = e[k] & 0xFFFFu, y = kBT ? ((e[k] >> 16) & 0x1FFFu) : (e[k] >> 16);
        const uint32_t tx0 = x >> 3, ty0 = y >> 3, bx = x & 7u, by = y & 7u;
        const uint32_t tidx = ty0 * c.Tw + tx0;
        const int hoff = (bx == 0u && tx0 > 0u) ? -1 : ((bx == 7u && tx0 + 1u < c.Tw) ? 1 : 0);
        const int voff = (by == 0u && ty0 > 0u) ? -(int)c.Tw : ((by == 7u && ty0 + 1u < c.Th) ? (int)c.Tw : 0);
        const uint4* const sp = c.thr4 + (size_t)(c.thr_sec + y * c.W + x) * 2;
        tc[k] = ldcg_u64(c.tiles + (c.plane_r + tidx));
        { const thr_sector ts = (K == 1) ? ldg_thr_early(sp) : ldg_thr(sp); Ta[k] = ts.a; Tb[k] = ts.b; }
        th[k] = 0ull; tv[k] = 0ull; td[k] = 0ull;
        if (hoff) th[k] = ldcg_u64(c.tiles + (c.plane_r + tidx + hoff));
        if (voff) tv[k] = ldcg_u64(c.tiles + (c.plane_r + tidx + voff));
        if (hoff && voff) td[k] = ldcg_u64(c.tiles + (c.plane_r + tidx + hoff + voff));
    }
    uint32_t cnt = 0;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const uint32_t bx = e[k] & 7u, by = (e[k] >> 16) & 7u;
        // rows y-1, y, y+1 of the cell's tile column (w3c) and of the horizontally adjacent one (w3h), one per byte
        const uint32_t selr = ((by + 7u) & 7u) | (by << 4) | (((by + 1u) & 7u) << 8);
        uint32_t w3c = __byte_perm((uint32_t)tc[k], (uint32_t)(tc[k] >> 32), selr) & 0xFFFFFFu;
        uint32_t w3h = __byte_perm((uint32_t)th[k], (uint32_t)(th[k] >> 32), selr) & 0xFFFFFFu;
        // row y-1 is row 7 of the tile above when by == 0, row y+1 is row 0 of the tile below when by == 7
        const uint32_t vc = (by == 0u) ? (uint32_t)(tv[k] >> 56) : (((uint32_t)tv[k] & 0xFFu) << 16);
        const uint32_t vh = (by == 0u) ? (uint32_t)(td[k] >> 56) : (((uint32_t)td[k] & 0xFFu) << 16);
        const uint32_t keep = (by == 0u) ? 0xFFFF00u : ((by == 7u) ? 0x00FFFFu : 0xFFFFFFu);
        w3c = (w3c & keep) | vc;                                     // tv = td = 0 unless by is 0 or 7
        w3h = (w3h & keep) | vh;
        // per byte: bit 0 = (x-1), bit 1 = x, bit 2 = (x+1)
        const uint32_t tcen = (w3c << 1) >> bx;
        const uint32_t mC = (bx == 0u) ? 0x060606u : ((bx == 7u) ? 0x030303u : 0x070707u);
        const uint32_t hb = (bx == 0u) ? ((w3h >> 7) & 0x010101u) : ((w3h << 2) & 0x040404u);
        win[k] = live[k] ? ((tcen & mC) | hb) : 0u;
        cnt += __popc(win[k]);
    }
    if (kBT) {
#pragma unroll
        for (int k = 0; k < K; ++k) {
            append_next(c, live[k] && (e[k] >> 29) != 0u, e[k] - (1u << 29));      // still burning next step
            e[k] &= 0x1FFFFFFFu;                                                   // the trial items are built from the coordinates
        }
    }
    uint32_t incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (c.lane >= (uint32_t)o) incl += v;
    }
    const uint32_t total = __shfl_sync(0xFFFFFFFFu, incl, 31);
    if (total == 0) return 0u;
    uint32_t qbase = 0;
    if (c.lane == 31) qbase = atoms_add(c.cntQ, total);
    qbase = __shfl_sync(0xFFFFFFFFu, qbase, 31);
    uint32_t pos = qbase + incl - cnt;
    if (qbase + total <= c.capQ_s) {                                  // warp-uniform: the whole batch fits in shared memory
#define FIRE_EMIT(bit, d, Tv) \
        if (w & (1u << (bit))) sts64(qa + 8u * __popc(w & ((1u << (bit)) - 1u)), base + item_delta(d), (Tv));
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const uint32_t w = win[k];
            const uint32_t base = e[k];
            const uint32_t qa = c.qs_addr + 8u * pos;
            FIRE_EMIT(0, 7, Tb[k].w)  FIRE_EMIT(1, 0, Ta[k].x)  FIRE_EMIT(2, 1, Ta[k].y)
            FIRE_EMIT(8, 6, Tb[k].z)  FIRE_EMIT(10, 2, Ta[k].z)
            FIRE_EMIT(16, 5, Tb[k].y) FIRE_EMIT(17, 4, Tb[k].x) FIRE_EMIT(18, 3, Ta[k].w)
            pos += __popc(w);
        }
#undef FIRE_EMIT
    } else {
#define FIRE_EMIT(bit, d, Tv) \
        if (w & (1u << (bit))) { \
            const uint32_t q = pos + __popc(w & ((1u << (bit)) - 1u)); \
            if (q < c.capQ_s) sts64(c.qs_addr + 8u * q, base + item_delta(d), (Tv)); \
            else __stcg(reinterpret_cast<uint2*>(c.spill + c.qg_off) + (q - c.capQ_s), make_uint2(base + item_delta(d), (Tv))); \
        }
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const uint32_t w = win[k];
            const uint32_t base = e[k];
            FIRE_EMIT(0, 7, Tb[k].w)  FIRE_EMIT(1, 0, Ta[k].x)  FIRE_EMIT(2, 1, Ta[k].y)
            FIRE_EMIT(8, 6, Tb[k].z)  FIRE_EMIT(10, 2, Ta[k].z)
            FIRE_EMIT(16, 5, Tb[k].y) FIRE_EMIT(17, 4, Tb[k].x) FIRE_EMIT(18, 3, Ta[k].w)
            pos += __popc(w);
        }
#undef FIRE_EMIT
    }
    return cnt;
}

// Philox keys and the per-step constants of rounds 0 and 1 (C-1; rounds 0 and 1 see (c1, c2) = (t, sim)).
struct philox_step {
    uint32_t rk0[10], rk1[10];   // round keys (rk0[0], rk0[1], rk1[1] are folded into the constants below)
    uint32_t x1, y1, a1l;
};

// Phase 2 for K units of 32 trials (units u0, u0 + ustride, ...; all of them exist: u * 32 < nQ), in two halves so
// that the caller can overlap the atomics of one pass with the arithmetic of the next:
//   trials_issue  : queue reads -> Philox -> compare -> atomicAnd on the susceptible plane (results left pending)
//   trials_resolve: the lane whose atomic saw the bit still set owns the new burning cell -> next frontier
constexpr int kMaxInFlight = 4;
struct pending_trials { uint32_t item[kMaxInFlight], bit[kMaxInFlight], old[kMaxInFlight]; };   // the first K entries are used

template <int K>
__device__ __forceinline__ void trials_issue(const step_ctx& c, const philox_step& ph, uint32_t u0, uint32_t ustride,
                                             pending_trials& pt)
{
    uint32_t T[K];
    if ((u0 + (uint32_t)(K - 1) * ustride + 1u) * 32u <= c.capQ_s) {                       // warp-uniform: all in shared memory
#pragma unroll
        for (int u = 0; u < K; ++u) {
            uint32_t j = (u0 + (uint32_t)u * ustride) * 32u + c.lane;
            const bool live = j < c.nQ;
            j = live ? j : c.nQ - 1u;                              // a lane past the end re-reads the last entry
            const uint2 it = lds64(c.qs_addr + 8u * j);
            pt.item[u] = it.x;
            T[u] = live ? it.y : 0u;                               // T = 0 never succeeds
        }
    } else {
#pragma unroll
        for (int u = 0; u < K; ++u) {
            uint32_t j = (u0 + (uint32_t)u * ustride) * 32u + c.lane;
            const bool live = j < c.nQ;
            j = live ? j : c.nQ - 1u;
            const uint2 it = (j < c.capQ_s) ? lds64(c.qs_addr + 8u * j) : __ldcg(reinterpret_cast<const uint2*>(c.spill + c.qg_off) + (j - c.capQ_s));
            pt.item[u] = it.x;
            T[u] = live ? it.y : 0u;
        }
    }
#pragma unroll
    for (int u = 0; u < K; ++u) {
        const uint32_t ty = pt.item[u] >> 16, tx = pt.item[u] & 0x1FFFu, d = (pt.item[u] >> 13) & 7u;
        const uint32_t cell = ty * c.W + tx;
        pt.bit[u] = ((ty & 3u) << 3) | (tx & 7u);
        const uint32_t widx = (((ty >> 3) * c.Tw + (tx >> 3)) << 1) | ((ty >> 2) & 1u);
        // round 0: (cell, t, sim, d >> 2) -> (r0c0, bl, hi(cell * M0) ^ (d >> 2) ^ k1, lo(cell * M0))
        uint32_t c3 = cell * kM0;
        uint32_t c2 = __umulhi(cell, kM0) ^ (d >> 2) ^ ph.rk1[0];
        // round 1: a = r0c0 * M0 (per step), b = c2 * M1
        uint32_t c0 = __umulhi(c2, kM1) ^ ph.x1;
        uint32_t c1 = c2 * kM1;
        c2 = ph.y1 ^ c3;
        c3 = ph.a1l;
#pragma unroll
        for (int r = 2; r < 10; ++r) {
            const uint64_t a = (uint64_t)c0 * kM0;
            const uint64_t b = (uint64_t)c2 * kM1;
            const uint32_t n0 = (uint32_t)(b >> 32) ^ c1 ^ ph.rk0[r];
            const uint32_t n2 = (uint32_t)(a >> 32) ^ c3 ^ ph.rk1[r];
            c1 = (uint32_t)b; c3 = (uint32_t)a; c0 = n0; c2 = n2;
        }
        const uint32_t lo = (d & 1u) ? c1 : c0, hi = (d & 1u) ? c3 : c2;
        const uint32_t rnd = (d & 2u) ? hi : lo;
        pt.old[u] = 0u;
        if (fire_trial(rnd, T[u])) {
            pt.old[u] = atomicAnd(reinterpret_cast<uint32_t*>(const_cast<uint64_t*>(c.tiles)) + (c.plane_w2 + widx), ~(1u << pt.bit[u]));
        }
    }
}

template <int K, bool kBT = false>
__device__ __forceinline__ void trials_resolve(const step_ctx& c, const pending_trials& pt)
{
    uint32_t fresh_mask[K];
    uint32_t n_fresh = 0;
#pragma unroll
    for (int u = 0; u < K; ++u) {
        fresh_mask[u] = __ballot_sync(0xFFFFFFFFu, (pt.old[u] >> pt.bit[u]) & 1u);     // old = 0 unless the trial succeeded
        n_fresh += __popc(fresh_mask[u]);
    }
    if (n_fresh == 0) return;                                      // warp-uniform
    uint32_t abase = 0;
    if (c.lane == 0) abase = atoms_add(c.cntA_next, n_fresh);
    abase = __shfl_sync(0xFFFFFFFFu, abase, 0);
    if (abase + n_fresh <= c.capA_s) {                             // warp-uniform: all new cells go to shared memory
#pragma unroll
        for (int u = 0; u < K; ++u) {
            uint32_t en = pt.item[u] & 0xFFFF1FFFu;
            const uint32_t a = c.an_addr + 4u * (abase + __popc(fresh_mask[u] & c.lt));
            if (fresh_mask[u] & (1u << c.lane)) {
                if (kBT) {
                    const uint32_t cell = (en >> 16) * c.W + (en & 0x1FFFu);
                    if (c.time_base) c.time_base[cell] = (int32_t)(c.t + 1u);                              // ignited by the transition t -> t + 1
                    en |= (uint32_t)__ldg(c.ktime + cell) << 29;                                           // burn time of its fuel - 1
                }
                sts32(a, en);
            }
            abase += __popc(fresh_mask[u]);
        }
    } else {
#pragma unroll
        for (int u = 0; u < K; ++u) {
            if (fresh_mask[u] & (1u << c.lane)) {
                const uint32_t pos = abase + __popc(fresh_mask[u] & c.lt);
                uint32_t en = pt.item[u] & 0xFFFF1FFFu;
                if (kBT) {
                    const uint32_t cell = (en >> 16) * c.W + (en & 0x1FFFu);
                    if (c.time_base) c.time_base[cell] = (int32_t)(c.t + 1u);
                    en |= (uint32_t)__ldg(c.ktime + cell) << 29;
                }
                if (pos < c.capA_s) sts32(c.an_addr + 4u * pos, en);
                else if (pos < c.capA) __stcg(c.spill + (c.an_off + (pos - c.capA_s)), en);
                else sts32(c.over, 1u);
            }
            abase += __popc(fresh_mask[u]);
        }
    }
}

// A pass of exactly k units (1 <= k <= KMAX), k warp-uniform: one specialised body per k, so that the last pass of a
// warp executes no code for units that do not exist.
template <int KMAX>
__device__ __forceinline__ void trials_issue_k(const step_ctx& c, const philox_step& ph, uint32_t u0, uint32_t ustride, int k,
                                               pending_trials& pt)
{
    if (KMAX >= 4 && k == 4) trials_issue<4>(c, ph, u0, ustride, pt);
    else if (KMAX >= 3 && k == 3) trials_issue<3>(c, ph, u0, ustride, pt);
    else if (KMAX >= 2 && k == 2) trials_issue<2>(c, ph, u0, ustride, pt);
    else trials_issue<1>(c, ph, u0, ustride, pt);
}
template <int KMAX, bool kBT = false>
__device__ __forceinline__ void trials_resolve_k(const step_ctx& c, int k, const pending_trials& pt)
{
    if (KMAX >= 4 && k == 4) trials_resolve<4, kBT>(c, pt);
    else if (KMAX >= 3 && k == 3) trials_resolve<3, kBT>(c, pt);
    else if (KMAX >= 2 && k == 2) trials_resolve<2, kBT>(c, pt);
    else if (k == 1) trials_resolve<1, kBT>(c, pt);
}

// ------------------------------------------------------------------------------------------------
// Fast kernel: one persistent CTA per simulation.
// Instantiated for a few (threads per CTA, CTAs per SM) bounds: the bound sets the register budget.
// kCellsInFlight / kTrialsInFlight: units of 32 burning cells (phase 1) / 32 trials (phase 2) a warp has in flight.
// ------------------------------------------------------------------------------------------------
template <int kMaxThreads, int kMinCtas, int kCellsInFlight, int kTrialsInFlight, bool kBT = false>
__global__ void __launch_bounds__(kMaxThreads, kMinCtas)
fire_propagate_kernel(const prop_params prm)
{
    extern __shared__ __align__(16) uint32_t smem[];
    // shared layout: trial queue (capQ_s x 8 B), frontier list 0, frontier list 1 (capA_s x 4 B each)
    uint32_t qs_addr = (uint32_t)__cvta_generic_to_shared(smem);
    asm volatile("" : "+r"(qs_addr));            // keep it in a register: ptxas would otherwise rebuild the window address at every use
    const uint32_t as_addr0 = qs_addr + 8u * prm.capQ_s, as_addr1 = as_addr0 + 4u * prm.capA_s;
    const size_t spill_per_cta = (size_t)2 * (prm.capQ - prm.capQ_s) + (size_t)2 * (prm.capA - prm.capA_s);
    // the host checks that the spill area has fewer than 2^32 words
    const uint32_t qg_off = (uint32_t)((size_t)blockIdx.x * spill_per_cta);
    const uint32_t ag_off0 = qg_off + 2u * (prm.capQ - prm.capQ_s), ag_off1 = ag_off0 + (prm.capA - prm.capA_s);

    __shared__ struct { unsigned int cntA[2], cntQ[2], over, sim; } s_ctl;      // counters in one block: one base address
    unsigned int (&s_cntA)[2] = s_ctl.cntA; unsigned int (&s_cntQ)[2] = s_ctl.cntQ;
    unsigned int& s_over = s_ctl.over; unsigned int& s_sim = s_ctl.sim;
    __shared__ unsigned long long s_trials;

    const int tid = threadIdx.x;
    const uint32_t warp = (uint32_t)tid >> 5, nwarps = blockDim.x >> 5;
    // floor(x / nwarps) = umulhi(x, inv) for every x < 2^32 / nwarps; 0 stands for nwarps = 1 (its reciprocal does not fit)
    const uint32_t inv_nwarps = nwarps > 1u ? 0xFFFFFFFFu / nwarps + 1u : 0u;

    step_ctx c;
    c.W = (uint32_t)prm.W; c.Tw = (uint32_t)prm.Tw; c.Th = (uint32_t)prm.Th; c.tiles = prm.tiles; c.thr4 = reinterpret_cast<const uint4*>(prm.thr);
    c.qs_addr = qs_addr; c.capQ_s = prm.capQ_s; c.capA_s = prm.capA_s; c.capA = prm.capA;
    c.spill = prm.spill; c.qg_off = qg_off;
    uint32_t cntA_addr = (uint32_t)__cvta_generic_to_shared(&s_cntA[0]);
    asm volatile("" : "+r"(cntA_addr));          // as for qs_addr; s_cntA[2], s_cntQ[2], s_over are laid out in this order
    const uint32_t cntQ_addr = cntA_addr + 8u;
    c.over = cntA_addr + 16u;
    c.lane = (uint32_t)tid & 31u; c.lt = lanemask_lt();
    c.ktime = prm.ktime; c.time_base = nullptr; c.t = 0u;

    for (;;) {
        __syncthreads();                       // the previous simulation's last reads of s_* are done
        if (tid == 0) s_sim = next_simulation(prm);
        __syncthreads();
        const uint32_t s = s_sim;
        if (s == 0xFFFFFFFFu) break;

        const int p = prm.sim_param[s];
        const int ix = prm.ignitions[2 * s], iy = prm.ignitions[2 * s + 1];
        const uint64_t seed = prm.seeds[s];
        const uint32_t sim = prm.sim_ids ? (uint32_t)prm.sim_ids[s] : s;
        c.plane_r = c.plane_w = s * (c.Tw * c.Th);             // the host checks that S * tiles fits 31 bits
        c.plane_w2 = c.plane_w << 1;
        asm volatile("" : "+r"(c.plane_w2));                  // once per simulation, used once per unit of trials
        bool valid = p >= 0 && p < prm.P && ix >= 0 && ix < prm.W && iy >= 0 && iy < prm.H;     // R-12
        if (valid) valid = (__ldg(prm.burnable + (size_t)iy * prm.Ww + (ix >> 5)) >> (ix & 31)) & 1u;
        c.thr_sec = valid ? (uint32_t)p * (c.W * (uint32_t)prm.H) : 0u;
        if (kBT) c.time_base = prm.out_time ? prm.out_time + (size_t)s * ((size_t)prm.W * prm.H) : nullptr;
        // the key is the same in every lane: a warp reduction leaves it in a UNIFORM register, and so are the round keys
        // derived from it (they then cost no per-thread registers)
        const uint32_t key_lo = __reduce_or_sync(0xFFFFFFFFu, (uint32_t)seed), key_hi = __reduce_or_sync(0xFFFFFFFFu, (uint32_t)(seed >> 32));
        // Philox round 0 multiplies the counter word `sim` by M1: the same product for every trial of the simulation
        const uint32_t bh = __umulhi(sim, kM1), bl = sim * kM1;

        if (tid == 0) {
            s_cntA[0] = valid ? 1u : 0u; s_cntA[1] = 0u; s_cntQ[0] = 0u; s_cntQ[1] = 0u;
            s_over = 0u; s_trials = 0ull;
            if (valid) {
                uint32_t e0 = ((uint32_t)iy << 16) | (uint32_t)ix;
                if (kBT) e0 |= (uint32_t)prm.ktime[(size_t)iy * prm.W + ix] << 29;
                if (kBT && c.time_base) c.time_base[(size_t)iy * prm.W + ix] = 0;
                if (prm.capA_s > 0) sts32(as_addr0, e0); else prm.spill[ag_off0] = e0;
                atomicAnd(reinterpret_cast<uint32_t*>(prm.tiles) + (((size_t)c.plane_w + (size_t)(iy >> 3) * c.Tw + (ix >> 3)) * 2 + ((iy >> 2) & 1)), ~(1u << (((iy & 3) << 3) | (ix & 7))));
            }
        }
        __syncthreads();

        uint32_t t = 0, my_trials = 0;
        c.nA = valid ? 1u : 0u;
        bool over = false;
        while (c.nA > 0 && (prm.max_steps == 0 || t < prm.max_steps)) {
            const uint32_t par = t & 1u;
            if (kBT) c.t = t;
            c.ac_addr = par ? as_addr1 : as_addr0; c.an_addr = par ? as_addr0 : as_addr1;
            c.ac_off = par ? ag_off1 : ag_off0; c.an_off = par ? ag_off0 : ag_off1;
            c.cntQ = cntQ_addr + 4u * par; c.cntA_next = cntA_addr + 4u * (par ^ 1u);

            // ---- phase 1: susceptible neighbours of the burning cells and their thresholds -> trial queue.
            // Units of 32 cells are dealt round-robin to the warps: full passes of kCellsInFlight units, then single units.
            {
                const uint32_t nU = (c.nA + 31u) >> 5;
                uint32_t u = warp;
                for (; u + (uint32_t)(kCellsInFlight - 1) * nwarps < nU; u += nwarps * kCellsInFlight)
                    my_trials += cells_pass<kCellsInFlight, kBT>(c, u, nwarps);
                for (; u < nU; u += nwarps) my_trials += cells_pass<1, kBT>(c, u, nwarps);
            }
            __syncthreads();
            c.nQ = s_cntQ[par];
            if (tid == 0) { s_cntA[par] = 0u; s_cntQ[par ^ 1u] = 0u; }    // next step's counters; nobody reads them now

            // ---- phase 2: one Bernoulli trial per lane-slot.  Philox4x32-10(counter = (cell, t, sim, d >> 2), key = seed),
            // word d & 3 (C-1).  Round keys are rebuilt once per step (they are dead during phase 1) and made
            // opaque so that they stay in registers.
            if (warp < ((c.nQ + 31u) >> 5)) {                   // warps without a unit of trials go straight to the barrier
                philox_step ph;
#pragma unroll
                for (int r = 0; r < 10; ++r) {
                    ph.rk0[r] = key_lo + (uint32_t)r * kW0;
                    ph.rk1[r] = key_hi + (uint32_t)r * kW1;
                }
                const uint32_t r0c0 = bh ^ t ^ ph.rk0[0];                          // c0 after round 0
                ph.a1l = r0c0 * kM0;                                               // round 1: c0 * M0
                ph.x1 = bl ^ ph.rk0[1];
                ph.y1 = __umulhi(r0c0, kM0) ^ ph.rk1[1];
                const uint32_t nU = (c.nQ + 31u) >> 5;
                uint32_t u = warp;
                // passes of up to kTrialsInFlight units, software-pipelined: the atomics of a pass are resolved after the
                // arithmetic of the next pass has been issued; the last pass of a warp has exactly the units that are left
                {
                    pending_trials prev;
                    bool have = false;
                    uint32_t left = (nU > u) ? (inv_nwarps ? __umulhi(nU - u + nwarps - 1u, inv_nwarps) : nU - u) : 0u;      // units of this warp: ceil((nU - u) / nwarps)
                    for (; left >= (uint32_t)kTrialsInFlight; left -= (uint32_t)kTrialsInFlight, u += nwarps * kTrialsInFlight) {
                        pending_trials cur;
                        trials_issue<kTrialsInFlight>(c, ph, u, nwarps, cur);
                        if (have) trials_resolve<kTrialsInFlight, kBT>(c, prev);
                        prev = cur; have = true;
                    }
                    if (left > 0u) {                               // the last, shorter pass: specialised by its exact size
                        pending_trials cur;
                        trials_issue_k<kTrialsInFlight>(c, ph, u, nwarps, (int)left, cur);
                        if (have) trials_resolve<kTrialsInFlight, kBT>(c, prev);
                        trials_resolve_k<kTrialsInFlight, kBT>(c, (int)left, cur);
                    } else if (have) {
                        trials_resolve<kTrialsInFlight, kBT>(c, prev);
                    }
                }
            }
            __syncthreads();
            ++t;
            if (s_over) { over = true; break; }       // written in phase 2 only, read after its closing barrier
            c.nA = s_cntA[par ^ 1u];
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


// The same first half for trials taken from a warp's own ring buffer (asynchronous-warp kernel): n <= 64 entries at `head`,
// as two interleaved units of 32 (the second one is skipped when n <= 32).
__device__ __forceinline__ void trials_issue_ring(const step_ctx& c, const philox_step& ph, uint32_t ring_addr, uint32_t head,
                                                  uint32_t n, uint32_t ring_mask, pending_trials& pt)
{
    uint32_t T[2];
#pragma unroll
    for (int u = 0; u < 2; ++u) {
        const bool live = c.lane + 32u * u < n;
        const uint2 it = lds64(ring_addr + 8u * ((head + (live ? c.lane + 32u * u : 0u)) & ring_mask));
        pt.item[u] = it.x;
        T[u] = live ? it.y : 0u;                                   // T = 0 never succeeds
        pt.old[u] = 0u; pt.bit[u] = 0u;
    }
#pragma unroll
    for (int u = 0; u < 2; ++u) {
        if (u == 1 && n <= 32u) break;                             // warp-uniform
        const uint32_t ty = pt.item[u] >> 16, tx = pt.item[u] & 0x1FFFu, d = (pt.item[u] >> 13) & 7u;
        const uint32_t cell = ty * c.W + tx;
        pt.bit[u] = ((ty & 3u) << 3) | (tx & 7u);
        const uint32_t widx = (((ty >> 3) * c.Tw + (tx >> 3)) << 1) | ((ty >> 2) & 1u);
        uint32_t c3 = cell * kM0;
        uint32_t c2 = __umulhi(cell, kM0) ^ (d >> 2) ^ ph.rk1[0];
        uint32_t c0 = __umulhi(c2, kM1) ^ ph.x1;
        uint32_t c1 = c2 * kM1;
        c2 = ph.y1 ^ c3;
        c3 = ph.a1l;
#pragma unroll
        for (int r = 2; r < 10; ++r) {
            const uint64_t a = (uint64_t)c0 * kM0;
            const uint64_t b = (uint64_t)c2 * kM1;
            const uint32_t n0 = (uint32_t)(b >> 32) ^ c1 ^ ph.rk0[r];
            const uint32_t n2 = (uint32_t)(a >> 32) ^ c3 ^ ph.rk1[r];
            c1 = (uint32_t)b; c3 = (uint32_t)a; c0 = n0; c2 = n2;
        }
        const uint32_t lo = (d & 1u) ? c1 : c0, hi = (d & 1u) ? c3 : c2;
        const uint32_t rnd = (d & 2u) ? hi : lo;
        if (fire_trial(rnd, T[u])) pt.old[u] = atomicAnd(reinterpret_cast<uint32_t*>(const_cast<uint64_t*>(c.tiles)) + (c.plane_w2 + widx), ~(1u << pt.bit[u]));
    }
}

// ------------------------------------------------------------------------------------------------
// Asynchronous-warp kernel: ONE block barrier per CA step.
// Two susceptible planes per simulation: step t READS plane t & 1 (exactly the state at the start of the step) and
// UPDATES plane (t + 1) & 1, which lags by the cells that are burning now; every burning cell first clears its own bit
// there ("catch-up", a fire-and-forget reduction), so that after the step the written plane is exactly the state at
// the start of step t + 1.  A successful trial's atomicAnd on the written plane still says who ignited the cell first.
// Because nothing read in a step is written in that step, there is no barrier between building trials and running
// them: every warp takes units of 32 burning cells, appends their trials to its OWN ring buffer in shared memory and
// runs them 32 at a time as soon as it has them; the loads of the next cell unit are in flight meanwhile.
// ------------------------------------------------------------------------------------------------
constexpr uint32_t kRingEntries = 512;             // per warp, 8 B each: one cell unit adds at most 256 trials to at most 31 left over

// With kCluster the kernel is launched as thread-block CLUSTERS of 2 or 4 CTAs (sm_90+), one cluster per simulation, for
// batches smaller than the GPU (config 5: 64 simulations of 4096 x 4096 on 148 SMs).  The state planes are in global memory
// (L2) and so are shared by construction; every CTA keeps the frontier list of the cells IT ignited in its own shared memory
// and the other CTAs of the cluster read it through distributed shared memory: of every list, CTA r runs the units
// u = (r + owner) mod size, so the work of a step is dealt evenly whoever owns the cells.  One cluster barrier per step.
__device__ __forceinline__ uint32_t cluster_ctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t cluster_nctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t cluster_map(uint32_t addr, uint32_t rank)
{
    uint32_t r; asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank)); return r;
}
__device__ __forceinline__ uint32_t ld_cluster32(uint32_t addr)
{
    uint32_t v; asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory"); return v;
}
__device__ __forceinline__ void st_cluster32(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared::cluster.u32 [%0], %1;" :: "r"(addr), "r"(v) : "memory");
}
template <bool kCluster>
__device__ __forceinline__ void team_sync()
{
    if (kCluster) asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
    else __syncthreads();
}
constexpr int kMaxClusterSize = 4;

template <int kMaxThreads, int kMinCtas, bool kCluster>
__global__ void __launch_bounds__(kMaxThreads, kMinCtas)
fire_propagate_async_kernel(const prop_params prm)
{
    extern __shared__ __align__(16) uint32_t smem[];
    const int tid = threadIdx.x;
    const uint32_t warp = (uint32_t)tid >> 5, nwarps = blockDim.x >> 5;
    const uint32_t crank = kCluster ? cluster_ctarank() : 0u, csize = kCluster ? cluster_nctarank() : 1u;
    // shared layout: per-warp trial rings, frontier list 0, frontier list 1
    uint32_t ring_addr = (uint32_t)__cvta_generic_to_shared(smem) + warp * (kRingEntries * 8u);
    asm volatile("" : "+r"(ring_addr));
    const uint32_t as_addr0 = (uint32_t)__cvta_generic_to_shared(smem) + nwarps * (kRingEntries * 8u), as_addr1 = as_addr0 + 4u * prm.capA_s;
    const size_t spill_per_cta = (size_t)2 * (prm.capQ - prm.capQ_s) + (size_t)2 * (prm.capA - prm.capA_s);
    // the host checks that the spill area has fewer than 2^32 words
    const uint32_t qg_off = (uint32_t)((size_t)blockIdx.x * spill_per_cta);
    const uint32_t ag_off0 = qg_off + 2u * (prm.capQ - prm.capQ_s), ag_off1 = ag_off0 + (prm.capA - prm.capA_s);

    __shared__ struct { unsigned int cntA[3], over, sim; } s_ctl;        // counters in one block: one base address
    unsigned int (&s_cntA)[3] = s_ctl.cntA; unsigned int& s_over = s_ctl.over; unsigned int& s_sim = s_ctl.sim;
    __shared__ unsigned long long s_trials;

    step_ctx c;
    c.W = (uint32_t)prm.W; c.Tw = (uint32_t)prm.Tw; c.Th = (uint32_t)prm.Th; c.tiles = prm.tiles; c.thr4 = reinterpret_cast<const uint4*>(prm.thr);
    c.capA_s = prm.capA_s; c.capA = prm.capA; c.capQ_s = 0u; c.qs_addr = 0u; c.spill = prm.spill; c.qg_off = qg_off; c.cntQ = 0u; c.nQ = 0u;
    uint32_t cntA_addr = (uint32_t)__cvta_generic_to_shared(&s_cntA[0]);
    asm volatile("" : "+r"(cntA_addr));          // as for ring_addr
    c.over = cntA_addr + 12u;
    c.lane = (uint32_t)tid & 31u; c.lt = lanemask_lt();
    const size_t nt = (size_t)c.Tw * c.Th;
    const uint32_t sim_addr = cntA_addr + 16u;
    const uint32_t trials_addr = (uint32_t)__cvta_generic_to_shared(&s_trials);

    for (;;) {
        team_sync<kCluster>();                 // the previous simulation's last (remote) reads of s_* are done
        if (tid == 0 && crank == 0) {
            const uint32_t nxt = next_simulation(prm);
            if (kCluster) { for (uint32_t j = 0; j < csize; ++j) st_cluster32(cluster_map(sim_addr, j), nxt); }
            else s_sim = nxt;
        }
        team_sync<kCluster>();
        const uint32_t s = s_sim;
        if (s == 0xFFFFFFFFu) break;
        const int p = prm.sim_param[s];
        const int ix = prm.ignitions[2 * s], iy = prm.ignitions[2 * s + 1];
        const uint64_t seed = prm.seeds[s];
        const uint32_t sim = prm.sim_ids ? (uint32_t)prm.sim_ids[s] : s;
        uint64_t* const plane0 = prm.tiles + (size_t)s * 2 * nt;
        const uint32_t plane0_t = s * 2u * (uint32_t)nt;
        bool valid = p >= 0 && p < prm.P && ix >= 0 && ix < prm.W && iy >= 0 && iy < prm.H;     // R-12
        if (valid) valid = (__ldg(prm.burnable + (size_t)iy * prm.Ww + (ix >> 5)) >> (ix & 31)) & 1u;
        c.thr_sec = valid ? (uint32_t)p * (c.W * (uint32_t)prm.H) : 0u;
        const uint32_t key_lo = __reduce_or_sync(0xFFFFFFFFu, (uint32_t)seed), key_hi = __reduce_or_sync(0xFFFFFFFFu, (uint32_t)(seed >> 32));
        const uint32_t bh = __umulhi(sim, kM1), bl = sim * kM1;

        if (tid == 0) {
            const bool seeded = valid && crank == 0u;              // the ignition cell belongs to the first CTA of the cluster
            s_cntA[0] = seeded ? 1u : 0u; s_cntA[1] = 0u; s_cntA[2] = 0u; s_over = 0u; s_trials = 0ull;
            if (seeded) {
                const uint32_t e0 = ((uint32_t)iy << 16) | (uint32_t)ix;
                if (prm.capA_s > 0) sts32(as_addr0, e0); else prm.spill[ag_off0] = e0;
                // the ignition is burnt at t = 0: cleared in plane 0 (read by step 0); plane 1 is caught up by step 0 itself
                atomicAnd(reinterpret_cast<uint32_t*>(plane0) + (((size_t)(iy >> 3) * c.Tw + (ix >> 3)) * 2 + ((iy >> 2) & 1)), ~(1u << (((iy & 3) << 3) | (ix & 7))));
            }
        }
        team_sync<kCluster>();

        uint32_t t = 0, my_trials = 0;
        uint32_t nA_of[kMaxClusterSize];                           // length of every CTA's current list; [0] is the only one without clusters
#pragma unroll
        for (int j = 0; j < kMaxClusterSize; ++j) nA_of[j] = 0u;
        nA_of[0] = valid ? 1u : 0u;
        uint32_t nA_total = nA_of[0];
        bool over = false;
        while (nA_total > 0 && (prm.max_steps == 0 || t < prm.max_steps)) {
            const uint32_t par = t & 1u;
            c.ac_addr = par ? as_addr1 : as_addr0; c.an_addr = par ? as_addr0 : as_addr1;
            c.ac_off = par ? ag_off1 : ag_off0; c.an_off = par ? ag_off0 : ag_off1;
            c.cntA_next = cntA_addr + 4u * ((t + 1u) % 3u);
            if (tid == 0) s_cntA[(t + 2u) % 3u] = 0u;             // read last at the start of step t - 1, appended to in step t + 1
            c.plane_r = plane0_t + par * (uint32_t)nt;                                        // read plane
            c.plane_w = plane0_t + (par ^ 1u) * (uint32_t)nt;                                 // written plane
            c.plane_w2 = c.plane_w << 1;

            philox_step ph;
#pragma unroll
            for (int r = 0; r < 10; ++r) { ph.rk0[r] = key_lo + (uint32_t)r * kW0; ph.rk1[r] = key_hi + (uint32_t)r * kW1; }
            const uint32_t r0c0 = bh ^ t ^ ph.rk0[0];
            ph.a1l = r0c0 * kM0; ph.x1 = bl ^ ph.rk0[1]; ph.y1 = __umulhi(r0c0, kM0) ^ ph.rk1[1];

            uint32_t head = 0, fill = 0;                           // this warp's ring: entries [head, head + fill) mod kRingEntries
            pending_trials prev; bool have = false;
#pragma unroll 1
            for (uint32_t j = 0; j < csize; ++j) {                 // the list of every CTA of the cluster (own list only without clusters)
            const uint32_t nA_j = kCluster ? nA_of[j] : nA_of[0];
            c.nA = nA_j;
            const uint32_t nU = (nA_j + 31u) >> 5;
            // where list j lives: the owner's shared memory (through the cluster window if it is not this CTA) and its global spill
            const bool own = !kCluster || j == crank;
            const uint32_t lst_addr = own ? c.ac_addr : cluster_map(c.ac_addr, j);
            const uint32_t lst_off = kCluster ? (uint32_t)((size_t)(blockIdx.x - crank + j) * spill_per_cta) + (c.ac_off - qg_off) : c.ac_off;
            const uint32_t u_first = kCluster ? ((crank + csize - (j % csize)) % csize) + csize * warp : warp;
            const uint32_t u_step = kCluster ? csize * nwarps : nwarps;
            for (uint32_t u = u_first; u < nU; u += u_step) {
                // ---- one unit of 32 burning cells: window, thresholds, catch-up, trials appended to the ring
                uint32_t i = u * 32u + c.lane;
                const bool live = i < c.nA;
                i = live ? i : c.nA - 1u;
                uint32_t e;
                if (i < c.capA_s) e = own ? lds32(lst_addr + 4u * i) : ld_cluster32(lst_addr + 4u * i);
                else e = __ldcg(c.spill + (lst_off + (i - c.capA_s)));
                const uint32_t x = e & 0xFFFFu, y = e >> 16;
                const uint32_t tx0 = x >> 3, ty0 = y >> 3, bx = x & 7u, by = y & 7u;
                const uint32_t tidx = ty0 * c.Tw + tx0;
                const int hoff = (bx == 0u && tx0 > 0u) ? -1 : ((bx == 7u && tx0 + 1u < c.Tw) ? 1 : 0);
                const int voff = (by == 0u && ty0 > 0u) ? -(int)c.Tw : ((by == 7u && ty0 + 1u < c.Th) ? (int)c.Tw : 0);
                const uint4* const sp = c.thr4 + (size_t)(c.thr_sec + y * c.W + x) * 2;
                const uint64_t tc = ldcg_u64(c.tiles + (c.plane_r + tidx));
                const thr_sector ts = ldg_thr(sp);
                const uint4 Ta = ts.a, Tb = ts.b;
                uint64_t th = 0ull, tv = 0ull, td = 0ull;
                if (hoff) th = ldcg_u64(c.tiles + (c.plane_r + tidx + hoff));
                if (voff) tv = ldcg_u64(c.tiles + (c.plane_r + tidx + voff));
                if (hoff && voff) td = ldcg_u64(c.tiles + (c.plane_r + tidx + hoff + voff));
                if (live) atomicAnd(reinterpret_cast<uint32_t*>(prm.tiles) + (((c.plane_w + tidx) << 1) | ((y >> 2) & 1u)), ~(1u << (((y & 3u) << 3) | bx)));      // catch-up (no return: RED)

                // while those loads are in flight: run the trials already in the ring
                while (fill >= 32u) {
                    const uint32_t n = fill >= 64u ? 64u : 32u;
                    pending_trials cur;
                    trials_issue_ring(c, ph, ring_addr, head, n, kRingEntries - 1u, cur);
                    if (have) trials_resolve<2>(c, prev);
                    prev = cur; have = true;
                    head = (head + n) & (kRingEntries - 1u); fill -= n;
                }

                const uint32_t selr = ((by + 7u) & 7u) | (by << 4) | (((by + 1u) & 7u) << 8);
                uint32_t w3c = __byte_perm((uint32_t)tc, (uint32_t)(tc >> 32), selr) & 0xFFFFFFu;
                uint32_t w3h = __byte_perm((uint32_t)th, (uint32_t)(th >> 32), selr) & 0xFFFFFFu;
                const uint32_t vc = (by == 0u) ? (uint32_t)(tv >> 56) : (((uint32_t)tv & 0xFFu) << 16);
                const uint32_t vh = (by == 0u) ? (uint32_t)(td >> 56) : (((uint32_t)td & 0xFFu) << 16);
                const uint32_t keep = (by == 0u) ? 0xFFFF00u : ((by == 7u) ? 0x00FFFFu : 0xFFFFFFu);
                w3c = (w3c & keep) | vc;
                w3h = (w3h & keep) | vh;
                const uint32_t tcen = (w3c << 1) >> bx;
                const uint32_t mC = (bx == 0u) ? 0x060606u : ((bx == 7u) ? 0x030303u : 0x070707u);
                const uint32_t hb = (bx == 0u) ? ((w3h >> 7) & 0x010101u) : ((w3h << 2) & 0x040404u);
                const uint32_t w = live ? ((tcen & mC) | hb) : 0u;
                const uint32_t cnt = __popc(w);
                uint32_t incl = cnt;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
                    if (c.lane >= (uint32_t)o) incl += v;
                }
                const uint32_t total = __shfl_sync(0xFFFFFFFFu, incl, 31);
                my_trials += cnt;
                const uint32_t pos = head + fill + incl - cnt;
                const uint32_t base = e;
#define FIRE_EMIT(bit, d, Tv) \
                if (w & (1u << (bit))) sts64(ring_addr + 8u * ((pos + __popc(w & ((1u << (bit)) - 1u))) & (kRingEntries - 1u)), base + item_delta(d), (Tv));
                FIRE_EMIT(0, 7, Tb.w)  FIRE_EMIT(1, 0, Ta.x)  FIRE_EMIT(2, 1, Ta.y)
                FIRE_EMIT(8, 6, Tb.z)  FIRE_EMIT(10, 2, Ta.z)
                FIRE_EMIT(16, 5, Tb.y) FIRE_EMIT(17, 4, Tb.x) FIRE_EMIT(18, 3, Ta.w)
#undef FIRE_EMIT
                fill += total;
                __syncwarp();
            }
            }
            // ---- the rest of the ring, last unit possibly partial
            while (fill > 0u) {
                const uint32_t n = fill < 64u ? fill : 64u;
                pending_trials cur;
                trials_issue_ring(c, ph, ring_addr, head, n, kRingEntries - 1u, cur);
                if (have) trials_resolve<2>(c, prev);
                prev = cur; have = true;
                head = (head + n) & (kRingEntries - 1u); fill -= n;
            }
            if (have) trials_resolve<2>(c, prev);
            team_sync<kCluster>();
            ++t;
            if (kCluster) {                                        // every CTA reads every CTA's flags and counters: all take the same decisions
                uint32_t ov[kMaxClusterSize];                      // all the remote loads first, then their uses: one round trip
#pragma unroll
                for (int j = 0; j < kMaxClusterSize; ++j) {
                    ov[j] = 0u; nA_of[j] = 0u;
                    if ((uint32_t)j < csize) {
                        ov[j] = ld_cluster32(cluster_map(c.over, (uint32_t)j));
                        nA_of[j] = ld_cluster32(cluster_map(cntA_addr + 4u * (t % 3u), (uint32_t)j));
                    }
                }
                const uint32_t any_over = ov[0] | ov[1] | ov[2] | ov[3];
                nA_total = nA_of[0] + nA_of[1] + nA_of[2] + nA_of[3];
                if (any_over) { over = true; break; }
            } else {
                if (s_over) { over = true; break; }
                nA_of[0] = s_cntA[t % 3u];
                nA_total = nA_of[0];
            }
        }

        if (my_trials) atomicAdd(&s_trials, (unsigned long long)my_trials);
        team_sync<kCluster>();
        if (tid == 0 && crank == 0u) {
            if (over) {
                prm.rescue_list[atomicAdd(prm.work_counter + 1, 1u)] = s;
            } else {
                unsigned long long trials = s_trials;
                if (kCluster)
                    for (uint32_t j = 1; j < csize; ++j)
                        trials += ((unsigned long long)ld_cluster32(cluster_map(trials_addr + 4u, j)) << 32) | ld_cluster32(cluster_map(trials_addr, j));
                prm.plane_sel[s] = t & 1u;                         // the plane that holds the final state
                if (prm.out_steps) prm.out_steps[s] = t;
                if (prm.out_trials) prm.out_trials[s] = trials;
            }
        }
    }
}


// ------------------------------------------------------------------------------------------------
// Plane set-up and tear-down around the fast kernel (pure streams).
//   fire_burnable_tiles_kernel : once per landscape, burnable bitmap -> tile layout
//   fire_init_tiles_kernel     : sus = burnable for every simulation of the batch
//   fire_finish_kernel         : burnt map (row-major bitmap) = burnable & ~sus
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
fire_burnable_tiles_kernel(const uint32_t* __restrict__ burnable, int H, int Ww, int Tw, int Th, uint64_t* __restrict__ out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= Tw * Th) return;
    const int ty = i / Tw, tx = i % Tw;
    uint64_t tile = 0ull;
    for (int r = 0; r < 8; ++r) {
        const int y = ty * 8 + r;
        if (y < H) tile |= (uint64_t)((burnable[(size_t)y * Ww + (tx >> 2)] >> ((tx & 3) * 8)) & 0xFFu) << (8 * r);
    }
    out[i] = tile;
}

__global__ void __launch_bounds__(256)
fire_init_tiles_kernel(const uint64_t* __restrict__ burnable_tiles, uint64_t* __restrict__ tiles, size_t nt, size_t nplanes)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t pl = blockIdx.y; pl < nplanes; pl += gridDim.y) {      // gridDim.y <= 65535 whatever the batch size
        uint64_t* const plane = tiles + pl * nt;
        if ((nt & 1) == 0) {
            const uint4* const b4 = reinterpret_cast<const uint4*>(burnable_tiles);
            uint4* const p4 = reinterpret_cast<uint4*>(plane);
            for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nt / 2; i += stride) p4[i] = __ldg(b4 + i);
        } else {
            for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nt; i += stride) plane[i] = __ldg(burnable_tiles + i);
        }
    }
}

// one thread per (tile row, bitmap word column): 4 tiles in (32 B), 8 words out (one per lattice row)
template <bool kFused>
__global__ void __launch_bounds__(256)
fire_finish_kernel(const uint32_t* __restrict__ burnable, const uint64_t* __restrict__ tiles, const uint32_t* __restrict__ plane_sel,
                   int planes, uint32_t* __restrict__ out_burned, int H, int Ww, int Tw, int Th, int S,
                   const uint32_t* __restrict__ fit_ref, uint32_t* __restrict__ fit_counts)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = i < Th * Ww;                                     // no early return: the fused counts are reduced per warp
    if (!kFused && !live) return;
    const int ty = live ? i / Ww : 0, wx = live ? i % Ww : 0;
    for (int s = blockIdx.y; s < S; s += gridDim.y) {                  // gridDim.y <= 65535 whatever the batch size
        uint32_t n_both = 0u, n_burnt = 0u;
        if (live) {
            const size_t plane = (size_t)s * planes + (planes > 1 ? (plane_sel[s] & 1u) : 0u);
            const uint64_t* const row = tiles + plane * Tw * Th + (size_t)ty * Tw;
            uint64_t tl[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) tl[k] = (4 * wx + k < Tw) ? __ldcs(reinterpret_cast<const unsigned long long*>(row + 4 * wx + k)) : 0ull;
            uint32_t* const out = out_burned + (size_t)s * H * Ww;
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                const int y = ty * 8 + r;
                if (y < H) {
                    uint32_t susw = 0u;
#pragma unroll
                    for (int k = 0; k < 4; ++k) susw |= (uint32_t)((tl[k] >> (8 * r)) & 0xFFull) << (8 * k);
                    const size_t wi = (size_t)y * Ww + wx;
                    const uint32_t bw = __ldg(burnable + wi) & ~susw;
                    out[wi] = bw;
                    if (kFused) { n_burnt += __popc(bw); n_both += __popc(bw & __ldg(fit_ref + wi)); }
                }
            }
        }
        if (kFused) {                                                  // Eq. 2's two counts, fused (fire_set_fused_counts)
            n_both = __reduce_add_sync(0xFFFFFFFFu, n_both);
            n_burnt = __reduce_add_sync(0xFFFFFFFFu, n_burnt);
            if ((threadIdx.x & 31) == 0 && (n_both | n_burnt)) {
                if (n_both) atomicAdd(fit_counts + 2 * (size_t)s, n_both);
                atomicAdd(fit_counts + 2 * (size_t)s + 1, n_burnt);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Launch order: simulations sorted by the mean contagion probability of their parameter vector,
// largest first (a counting sort on a 10-bit key).  Burn sizes are heavy-tailed
// (PAPER.md:135, :211): starting the large fires first lets the small ones fill the tail of the launch.
// ------------------------------------------------------------------------------------------------
constexpr int kOrderBuckets = 1024;
__global__ void __launch_bounds__(1024)
fire_order_kernel(const int32_t* __restrict__ sim_param, const float* __restrict__ param_mean, int S, int P, float scale, uint32_t* __restrict__ order)
{
    __shared__ unsigned int hist[kOrderBuckets];
    __shared__ unsigned int start[kOrderBuckets];
    const int tid = threadIdx.x;
    for (int b = tid; b < kOrderBuckets; b += blockDim.x) hist[b] = 0u;
    __syncthreads();
    auto bucket_of = [&](int s) -> int {
        const int p = sim_param[s];
        float m = (p >= 0 && p < P) ? param_mean[p] * scale : 0.0f;
        m = fminf(fmaxf(m, 0.0f), 1.0f);
        return (kOrderBuckets - 1) - (int)(m * (float)(kOrderBuckets - 1));     // bucket 0 = largest mean
    };
    for (int s = tid; s < S; s += blockDim.x) atomicAdd(&hist[bucket_of(s)], 1u);
    __syncthreads();
    if (tid == 0) {
        unsigned int acc = 0u;
        for (int b = 0; b < kOrderBuckets; ++b) { start[b] = acc; acc += hist[b]; }
    }
    __syncthreads();
    // order inside a bucket is whatever the atomics give: it only decides scheduling, never results
    for (int s = tid; s < S; s += blockDim.x) order[atomicAdd(&start[bucket_of(s)], 1u)] = (uint32_t)s;
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

// fire_set_fused_counts for a rescued simulation: the finish kernel counted the fast kernel's half-done plane, so the rescue
// kernel OVERWRITES (I, N*) with the counts of the map it has just written.  Called by every thread of the CTA.
__device__ __forceinline__ void rescue_fused_counts(const prop_params& prm, const uint32_t* burned, uint32_t s, unsigned int* s_fit)
{
    const size_t nw = (size_t)prm.H * prm.Ww;
    if (threadIdx.x == 0) { s_fit[0] = 0u; s_fit[1] = 0u; }
    __syncthreads();                                  // also orders the block's own writes to `burned` before the reads below
    uint32_t n_both = 0u, n_burnt = 0u;
    for (size_t w = threadIdx.x; w < nw; w += blockDim.x) {
        const uint32_t bw = __ldcg(burned + w);
        n_burnt += __popc(bw);
        n_both += __popc(bw & __ldg(prm.fit_ref + w));
    }
    n_both = __reduce_add_sync(0xFFFFFFFFu, n_both);
    n_burnt = __reduce_add_sync(0xFFFFFFFFu, n_burnt);
    if ((threadIdx.x & 31) == 0) { atomicAdd(&s_fit[0], n_both); atomicAdd(&s_fit[1], n_burnt); }
    __syncthreads();
    if (threadIdx.x == 0) { prm.fit_counts[2 * (size_t)s] = s_fit[0]; prm.fit_counts[2 * (size_t)s + 1] = s_fit[1]; }
}

__global__ void __launch_bounds__(256)
fire_propagate_rescue_kernel(const prop_params prm, uint32_t* planes)
{
    __shared__ int s_y0, s_y1;
    __shared__ unsigned long long s_trials;
    __shared__ unsigned int s_fit[2];
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
                        const uint32_t T = __ldg(thr + (size_t)(c - (uint32_t)(fire_dy(d) * W + fire_dx(d))) * 8 + d);   // slot d of the source cell
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
        if (prm.fit_counts) rescue_fused_counts(prm, burned, s, s_fit);
        __syncthreads();
        if (tid == 0) {
            if (prm.out_steps) prm.out_steps[s] = t;
            if (prm.out_trials) prm.out_trials[s] = s_trials;
        }
        __syncthreads();
    }
}

// The rescue kernel for fuel-dependent burn-out times (R-21).  planes: [gridDim.x][kmax + 1][H*Ww], a ring of "ignited by the
// transition into state tau" planes, all-zero on entry and on exit; a cell is active at step t iff it ignited at tau = t - j with
// burn time > j, i.e. active(t) = OR_j ring[(t - j) mod (kmax + 1)] & gt[j] with gt[0] = everything, gt[j] = prm.gt_planes[j - 1].
__device__ __forceinline__ uint32_t active_word(const prop_params& prm, const uint32_t* ring, size_t nw, uint32_t t, int y, int wx)
{
    if ((unsigned)y >= (unsigned)prm.H || (unsigned)wx >= (unsigned)prm.Ww) return 0u;
    const size_t wi = (size_t)y * prm.Ww + wx;
    const uint32_t R1 = (uint32_t)prm.kmax + 1u;
    uint32_t a = __ldcg(ring + (size_t)(t % R1) * nw + wi);
    for (uint32_t j = 1; j < (uint32_t)prm.kmax && j <= t; ++j)
        a |= __ldcg(ring + (size_t)((t - j) % R1) * nw + wi) & __ldg(prm.gt_planes + (size_t)(j - 1) * nw + wi);
    return a;
}

__global__ void __launch_bounds__(256)
fire_propagate_rescue_bt_kernel(const prop_params prm, uint32_t* planes)
{
    __shared__ int s_y0, s_y1;
    __shared__ unsigned long long s_trials;
    __shared__ unsigned int s_fit[2];
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int W = prm.W, H = prm.H, Ww = prm.Ww;
    const size_t nw = (size_t)H * Ww;
    const uint32_t R1 = (uint32_t)prm.kmax + 1u;
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
        uint32_t* const ring = planes + (size_t)blockIdx.x * R1 * nw;

        for (size_t w = tid; w < nw; w += nthr) burned[w] = 0u;      // the fast kernel left it half-done
        if (prm.out_time) for (size_t c = tid; c < (size_t)W * H; c += nthr) prm.out_time[(size_t)s * W * H + c] = -1;
        if (tid == 0) { s_y0 = iy; s_y1 = iy; s_trials = 0ull; }
        __syncthreads();
        if (tid == 0) {
            burned[(size_t)iy * Ww + (ix >> 5)] = 1u << (ix & 31);
            ring[(size_t)iy * Ww + (ix >> 5)] = 1u << (ix & 31);      // ignited "by the transition into state 0"
            if (prm.out_time) prm.out_time[(size_t)s * W * H + (size_t)iy * W + ix] = 0;
        }
        __syncthreads();

        uint32_t t = 0;
        unsigned long long my_trials = 0;
        int burning = 1;
        while (burning && (prm.max_steps == 0 || t < prm.max_steps)) {
            const int ylo = max(s_y0 - 1, 0), yhi = min(s_y1 + 1, H - 1);
            const int nwords = (yhi - ylo + 1) * Ww;
            uint32_t* const nxt = ring + (size_t)((t + 1u) % R1) * nw;
            int any_new = 0, ny0 = H, ny1 = -1;
            for (int idx = tid; idx < nwords; idx += nthr) {
                const int y = ylo + idx / Ww, wx = idx % Ww;
                const uint32_t uL = active_word(prm, ring, nw, t, y - 1, wx - 1), uC = active_word(prm, ring, nw, t, y - 1, wx),
                               uR = active_word(prm, ring, nw, t, y - 1, wx + 1);
                const uint32_t mL = active_word(prm, ring, nw, t, y, wx - 1), mC = active_word(prm, ring, nw, t, y, wx),
                               mR = active_word(prm, ring, nw, t, y, wx + 1);
                const uint32_t dL = active_word(prm, ring, nw, t, y + 1, wx - 1), dC = active_word(prm, ring, nw, t, y + 1, wx),
                               dR = active_word(prm, ring, nw, t, y + 1, wx + 1);
                uint32_t src[8];
                src[0] = dC;
                src[1] = (dC << 1) | (dL >> 31);
                src[2] = (mC << 1) | (mL >> 31);
                src[3] = (uC << 1) | (uL >> 31);
                src[4] = uC;
                src[5] = (uC >> 1) | (uR << 31);
                src[6] = (mC >> 1) | (mR << 31);
                src[7] = (dC >> 1) | (dR << 31);
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
                        const uint32_t T = __ldg(thr + (size_t)(c - (uint32_t)(fire_dy(d) * W + fire_dx(d))) * 8 + d);
                        hit |= fire_trial(fire_rnd(key_lo, key_hi, sim, t, c, d), T);
                    }
                    if (hit) {
                        fresh |= 1u << bx;
                        if (prm.out_time) prm.out_time[(size_t)s * W * H + c] = (int32_t)(t + 1u);
                    }
                }
                nxt[wi] = fresh;                      // always written: this ring slot held the ignitions of kmax + 1 steps ago
                if (fresh) { any_new = 1; ny0 = min(ny0, y); ny1 = max(ny1, y); }
            }
            __syncthreads();
            int still = any_new;
            for (int idx = tid; idx < nwords; idx += nthr) {
                const size_t wi = (size_t)ylo * Ww + idx;
                const uint32_t f = __ldcg(nxt + wi);
                if (f) burned[wi] |= f;
                if (!still && active_word(prm, ring, nw, t + 1u, ylo + idx / Ww, idx % Ww)) still = 1;    // cells that keep burning
            }
            if (any_new) { atomicMin(&s_y0, ny0); atomicMax(&s_y1, ny1); }
            burning = __syncthreads_or(still);
            ++t;
        }
        {   // leave the whole ring all-zero for the next simulation
            const int ylo = max(s_y0 - 1, 0), yhi = min(s_y1 + 1, H - 1);
            const size_t lo = (size_t)ylo * Ww, n = (size_t)(yhi - ylo + 1) * Ww;
            for (uint32_t r = 0; r < R1; ++r)
                for (size_t w = tid; w < n; w += nthr) ring[(size_t)r * nw + lo + w] = 0u;
        }
        if (my_trials) atomicAdd(&s_trials, my_trials);
        if (prm.fit_counts) rescue_fused_counts(prm, burned, s, s_fit);
        __syncthreads();
        if (tid == 0) {
            if (prm.out_steps) prm.out_steps[s] = t;
            if (prm.out_trials) prm.out_trials[s] = s_trials;
        }
        __syncthreads();
    }
}

// fire_set_burn_time: per-cell burn time - 1 from the vegetation class, and the bitmaps "burn time > j + 1" of the rescue kernel
struct burn_table { uint8_t k[256]; };
__global__ void __launch_bounds__(256)
fire_ktime_kernel(const uint8_t* __restrict__ veg, const burn_table tab, int W, int H, int Ww, int kmax, uint8_t* __restrict__ ktime,
                  uint32_t* __restrict__ gt_planes)
{
    const size_t warp = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;      // one warp per bitmap word
    const int lane = threadIdx.x & 31;
    const size_t nw = (size_t)H * Ww;
    if (warp >= nw) return;
    const int y = (int)(warp / Ww), x = (int)(warp % Ww) * 32 + lane;
    uint32_t k1 = 0u;
    if (x < W) {
        const size_t c = (size_t)y * W + x;
        const uint8_t v = veg[c];
        k1 = v ? (uint32_t)tab.k[v] - 1u : 0u;
        ktime[c] = (uint8_t)k1;
    }
    for (int j = 1; j < kmax; ++j) {
        const uint32_t word = __ballot_sync(0xFFFFFFFFu, k1 >= (uint32_t)j);            // burn time > j
        if (lane == 0) gt_planes[(size_t)(j - 1) * nw + warp] = word;
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

extern "C" int fire_set_schedule(fire_landscape* L, int32_t mode)
{
    if (L == nullptr || mode < 0) return FIRE_EINVAL;
    L->schedule = mode & 1;
    return FIRE_OK;
}

extern "C" int fire_set_burn_time(fire_landscape* L, const uint8_t* burn_time_host, int32_t n_classes, void* stream)
{
    if (L == nullptr || n_classes < 0 || n_classes > 256 || (n_classes > 0 && burn_time_host == nullptr)) return FIRE_EINVAL;
    if (L->sticky) return L->sticky;
    burn_table tab;
    int kmax = 1;
    for (int v = 0; v < 256; ++v) {
        int k = v < n_classes ? (int)burn_time_host[v] : 1;
        if (k == 0) k = 1;
        if (k > 8) return FIRE_EINVAL;
        tab.k[v] = (uint8_t)k;
        if (v > 0 && k > kmax) kmax = k;
    }
    if (kmax == 1) { L->burn_kmax = 1; return FIRE_OK; }          // the base model: nothing to keep
    fire_device_guard g(L->device);
    if (!g.ok) return FIRE_ECUDA;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nw = (size_t)L->H * L->Ww;
    if (L->ktime == nullptr || L->gt_capacity < nw * 4 * 7) {
        FIRE_CUDA_TRY(L, cudaStreamSynchronize(st));
        size_t cap = 0;
        if (L->ktime == nullptr) { int rc = fire_reserve(L, (void**)&L->ktime, &cap, L->cells); if (rc != FIRE_OK) return rc; }
        int rc = fire_reserve(L, (void**)&L->gt_planes, &L->gt_capacity, nw * 4 * 7);
        if (rc != FIRE_OK) return rc;
    }
    fire_ktime_kernel<<<(unsigned)((nw * 32 + 255) / 256), 256, 0, st>>>(L->veg_class, tab, L->W, L->H, L->Ww, kmax, L->ktime, L->gt_planes);
    FIRE_CUDA_TRY(L, cudaGetLastError());
    L->launches += 1;
    L->burn_kmax = kmax;
    return FIRE_OK;
}

extern "C" int fire_set_fused_counts(fire_landscape* L, const uint32_t* reference, uint32_t* out_counts)
{
    if (L == nullptr || (reference == nullptr) != (out_counts == nullptr)) return FIRE_EINVAL;      // set or cleared together
    L->fit_ref = reference;
    L->fit_counts = out_counts;
    return FIRE_OK;
}

extern "C" int fire_set_time_output(fire_landscape* L, int32_t* out_time)
{
    if (L == nullptr) return FIRE_EINVAL;
    L->out_time = out_time;
    return FIRE_OK;
}

extern "C" int fire_set_kernel(fire_landscape* L, int32_t family)
{
    if (L == nullptr || family < 0 || family > 4) return FIRE_EINVAL;
    L->kernel_family = family;
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
    // default: 4 CTAs of 256 threads per SM when there are enough simulations to fill them (16 CTAs of 128 threads with the
    // 32-register instantiation for very large batches on small lattices, whose fronts are a few dozen cells: config 4),
    // else fewer and wider CTAs so that a small batch of large fires still uses whole SMs
    int threads = L->threads_per_cta, per_sm = L->ctas_per_sm;
    if (threads == 0 && per_sm == 0) {
        if ((long long)S >= 16ll * L->num_sms && L->cells <= (size_t)512 * 512) { threads = 128; per_sm = 16; }   // small lattice = short fronts
        else if ((long long)S >= 4ll * L->num_sms) { threads = 256; per_sm = 4; }
        else if ((long long)S >= 2ll * L->num_sms) { threads = 512; per_sm = 2; }
        else { threads = 1024; per_sm = 1; }
    } else {
        if (threads == 0) threads = 256;
        if (per_sm == 0) per_sm = (1024 / threads) > 0 ? (1024 / threads) : 1;
    }
    // kernel family (fire_set_kernel): 1 = two-phase kernel (one state plane, two block barriers per step), 2 = asynchronous-warp
    // kernel (two state planes, one barrier per step, per-warp trial rings), 3 / 4 = the same as thread-block clusters of 2 / 4
    // CTAs per simulation; 0 = the two-phase kernel for batches that fill the GPU with 256-thread CTAs, the asynchronous-warp
    // kernel for small batches of large fires (wide CTAs, lattices of 2048 x 2048 or more), as clusters when the batch is smaller
    // than half the GPU
    // fuel-dependent burn-out times (fire_set_burn_time) are a variant of the two-phase kernel only
    const bool bt = L->burn_kmax > 1 || L->out_time != nullptr;         // ignition times are written by the same variant
    // (measured on one simulation of config 3 alone on the GPU: 2.6 us per step with the two-phase kernel at 1024 threads, 3.2 with
    // the asynchronous-warp kernel, 5.0-5.6 as a cluster -- a cluster barrier costs about 2 us; on config 5, whose fronts are
    // thousands of cells long, 89.6 / 85.0 / 64.2 ms: the wide families pay off on large lattices only)
    const bool big_lattice = L->cells >= (size_t)2048 * 2048;
    const bool async = !bt && (L->kernel_family >= 2 || (L->kernel_family == 0 && threads >= 512 && L->threads_per_cta == 0 && big_lattice));
    int cluster = !async ? 1 : (L->kernel_family == 3 ? 2 : (L->kernel_family == 4 ? 4 : 1));
    if (L->kernel_family == 0 && async && threads == 1024)
        cluster = (long long)S * 4 <= L->num_sms ? 4 : ((long long)S * 2 <= L->num_sms ? 2 : 1);
    // the cluster variant needs 72 registers: at 1,024 threads (64) it spills inside the unit loop; 28 warps without spills are
    // faster than 32 with (config 5: 65.4 -> 62.5 ms; 640 ... 896 threads all within 1 %)
    if (L->kernel_family == 0 && cluster > 1 && threads == 1024) threads = 896;
    const long long resident = (long long)L->num_sms * per_sm / cluster;         // simulations in flight
    const int grid = (int)((long long)S < resident ? S : (resident < 1 ? 1 : resident)) * cluster;
    const int planes = async ? 2 : 1;
    prop_params prm;
    uint32_t capA = L->list_capacity ? (uint32_t)L->list_capacity : 0u;
    if (capA == 0) {
        // generous: the burning front of a W x H lattice is a curve, not an area
        size_t want = (size_t)8 * (size_t)(L->W + L->H);
        if (want < 8192) want = 8192;
        if (want > L->cells) want = L->cells;
        capA = (uint32_t)want;
    }
    if (capA < 1) capA = 1;
    uint32_t capA_s = 1536u;                                   // 24 B of shared memory per entry (two lists + 2 queue slots)
    {
        const uint32_t fit = (uint32_t)((180u * 1024u) / ((uint32_t)per_sm * 24u)) & ~127u;
        if (capA_s > fit) capA_s = fit < 128u ? 128u : fit;
    }
    if (L->list_shared) capA_s = (uint32_t)L->list_shared;
    if (capA_s > capA) capA_s = capA;
    prm.capA_s = capA_s; prm.capA = capA;
    prm.capQ = 8u * capA;
    prm.capQ_s = 2u * capA_s;                                  // default: 1536-cell lists + 3072-trial queue = 36 KiB per CTA
    const size_t smem = async ? ((size_t)(threads / 32) * kRingEntries * 8 + (size_t)2 * prm.capA_s * sizeof(uint32_t))
                              : ((size_t)2 * prm.capA_s + (size_t)2 * prm.capQ_s) * sizeof(uint32_t);
    if (prm.capQ_s > prm.capQ) prm.capQ_s = prm.capQ;
    if (smem > (size_t)227 * 1024 - 1024) return FIRE_EINVAL;

    // ---- scratch owned by the handle (grow-only; growing waits for the stream first: see fire.h)
    const size_t spill_per_list_set = (size_t)2 * (prm.capQ - prm.capQ_s) + (size_t)2 * (prm.capA - prm.capA_s);   // per CTA
    const size_t spill_sets = (size_t)grid;
    const size_t spill_bytes = spill_per_list_set * spill_sets * 4 + 16;
    if (spill_per_list_set * spill_sets >= ((size_t)1 << 32)) return FIRE_EINVAL;   // spill slots are addressed by 32-bit word offsets
    const size_t nw = (size_t)L->H * L->Ww;
    const size_t nt = (size_t)L->Tw * L->Th;
    const int kmax = L->burn_kmax > 1 ? L->burn_kmax : 1;
    const size_t rescue_bytes = nw * 4 * (bt ? (size_t)kmax + 1 : 2) * kRescueCtas;
    if (nt * (size_t)S * planes >= ((size_t)1 << 31)) return FIRE_EINVAL;   // planes are addressed by 32-bit tile offsets: split the batch
    const size_t tiles_bytes = nt * 8 * (size_t)S * planes;
    if (L->status_capacity < (size_t)2 * S || L->spill_capacity < spill_bytes || L->rescue_capacity < rescue_bytes ||
        L->tiles_capacity < tiles_bytes || L->order_capacity < (size_t)S * 4 || L->burnable_tiles == nullptr) {
        FIRE_CUDA_TRY(L, cudaStreamSynchronize(st));
        size_t cap_bytes = L->status_capacity * 4;
        int rc = fire_reserve(L, (void**)&L->status, &cap_bytes, (size_t)2 * S * 4);     // rescue list [S] + plane selector [S]
        if (rc != FIRE_OK) return rc;
        L->status_capacity = cap_bytes / 4;
        rc = fire_reserve(L, (void**)&L->spill, &L->spill_capacity, spill_bytes);
        if (rc != FIRE_OK) return rc;
        rc = fire_reserve(L, (void**)&L->tiles, &L->tiles_capacity, tiles_bytes);
        if (rc != FIRE_OK) return rc;
        rc = fire_reserve(L, (void**)&L->order, &L->order_capacity, (size_t)S * 4);
        if (rc != FIRE_OK) return rc;
        if (L->rescue_capacity < rescue_bytes) {
            rc = fire_reserve(L, (void**)&L->rescue_planes, &L->rescue_capacity, rescue_bytes);
            if (rc != FIRE_OK) return rc;
            FIRE_CUDA_TRY(L, cudaMemsetAsync(L->rescue_planes, 0, L->rescue_capacity, st));
        }
        if (L->burnable_tiles == nullptr) {
            size_t cap = 0;
            rc = fire_reserve(L, (void**)&L->burnable_tiles, &cap, nt * 8);
            if (rc != FIRE_OK) return rc;
            fire_burnable_tiles_kernel<<<(unsigned)((nt + 255) / 256), 256, 0, st>>>(L->burnable, L->H, L->Ww, L->Tw, L->Th, L->burnable_tiles);
            FIRE_CUDA_TRY(L, cudaGetLastError());
            L->launches += 1;
        }
    }

    prm.burnable = L->burnable; prm.thr = L->thr;
    prm.ignitions = ignitions; prm.sim_param = sim_param; prm.seeds = seeds; prm.sim_ids = sim_ids;
    prm.tiles = L->tiles; prm.plane_sel = L->status + S;
    prm.out_burned = out_burned; prm.out_steps = out_steps; prm.out_trials = (unsigned long long*)out_trials;
    prm.work_counter = L->work_counter; prm.rescue_list = L->status; prm.spill = L->spill;
    prm.S = S; prm.P = L->P; prm.W = L->W; prm.H = L->H; prm.Ww = L->Ww; prm.Tw = L->Tw; prm.Th = L->Th; prm.num_sms = L->num_sms;
    prm.max_steps = max_steps;
    if (bt && (L->ktime == nullptr || L->burn_kmax <= 1)) {               // ignition times without burn times: every cell burns one step
        if (L->ktime == nullptr) {
            FIRE_CUDA_TRY(L, cudaStreamSynchronize(st));
            size_t cap = 0;
            int rc = fire_reserve(L, (void**)&L->ktime, &cap, L->cells);
            if (rc != FIRE_OK) return rc;
        }
        FIRE_CUDA_TRY(L, cudaMemsetAsync(L->ktime, 0, L->cells, st));
    }
    prm.ktime = bt ? L->ktime : nullptr; prm.gt_planes = bt ? L->gt_planes : nullptr; prm.kmax = kmax;
    prm.out_time = L->out_time;
    prm.fit_ref = L->fit_ref;
    prm.fit_counts = L->fit_counts;
    if (L->fit_counts) FIRE_CUDA_TRY(L, cudaMemsetAsync(L->fit_counts, 0, (size_t)S * 2 * sizeof(uint32_t), st));
    if (L->out_time) FIRE_CUDA_TRY(L, cudaMemsetAsync(L->out_time, 0xFF, (size_t)S * L->cells * sizeof(int32_t), st));      // -1 = never ignited

    // ---- launch order: largest expected fires first (only matters when there are more simulations than resident ones)
    prm.order = nullptr;
    if (S > grid / cluster && L->param_mean != nullptr && L->schedule == 0) {
        fire_order_kernel<<<1, 1024, 0, st>>>(sim_param, L->param_mean, S, L->P, 1.0f / ((float)L->cells * 8.0f), L->order);
        FIRE_CUDA_TRY(L, cudaGetLastError());
        L->launches += 1;
        prm.order = L->order;
    }

    // ---- planes: sus = burnable (tile layout), then the simulations, then burnt = burnable & ~sus (row-major bitmap)
    {
        const size_t units = (nt & 1) ? nt : nt / 2;
        unsigned chunks = (unsigned)((units + 256 * 4 - 1) / (256 * 4));
        if (chunks < 1) chunks = 1;
        if (chunks > 64) chunks = 64;
        const size_t nplanes = (size_t)S * planes;
        fire_init_tiles_kernel<<<dim3(chunks, (unsigned)(nplanes < 65535 ? nplanes : 65535)), 256, 0, st>>>(L->burnable_tiles, L->tiles, nt, nplanes);
        FIRE_CUDA_TRY(L, cudaGetLastError());
    }
    FIRE_CUDA_TRY(L, cudaMemsetAsync(L->work_counter, 0, 4 * sizeof(unsigned int), st));
    if (async) FIRE_CUDA_TRY(L, cudaMemsetAsync(L->status + S, 0, (size_t)S * 4, st));
    // instantiations differ in their register budget only (threads <= kMaxThreads is the one hard constraint)
    void (*kernel)(const prop_params) = nullptr;
    if (async && cluster > 1) kernel = threads <= 256 ? fire_propagate_async_kernel<256, 4, true> : (threads <= 512 ? fire_propagate_async_kernel<512, 2, true> : (threads <= 896 ? fire_propagate_async_kernel<896, 1, true> : fire_propagate_async_kernel<1024, 1, true>));
    else if (async) kernel = threads <= 256 ? fire_propagate_async_kernel<256, 4, false> : (threads <= 512 ? fire_propagate_async_kernel<512, 2, false> : fire_propagate_async_kernel<1024, 1, false>);
    else if (bt) kernel = threads <= 256 ? fire_propagate_kernel<256, 4, 2, 4, true>
                                         : (threads <= 512 ? fire_propagate_kernel<512, 2, 2, 4, true> : fire_propagate_kernel<1024, 1, 2, 4, true>);
    else kernel = threads <= 256 ? (per_sm <= 4 ? fire_propagate_kernel<256, 4, 2, 4> : fire_propagate_kernel<256, 8, 1, 2>)
                                 : (threads <= 512 ? fire_propagate_kernel<512, 2, 2, 4> : fire_propagate_kernel<1024, 1, 2, 4>);
    if (smem + 1024 > 48 * 1024)                     // dynamic + static shared memory beyond the default limit
        FIRE_CUDA_TRY(L, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    {   // ask for just the shared memory the resident CTAs need, so that the rest of the 228 KB stays L1
        int pct = (int)(((size_t)per_sm * (smem + 1024 + 256) * 100 + 228 * 1024 - 1) / (228 * 1024));   // + 1 KiB reserved per CTA + static shared memory
        if (pct > 100) pct = 100;
        FIRE_CUDA_TRY(L, cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, pct));
    }
    const bool prof = L->prof_enabled && L->prof_count < 64;
    if (prof) FIRE_CUDA_TRY(L, cudaEventRecord(L->prof_ev[2 * L->prof_count], st));
    if (cluster > 1) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)threads); cfg.dynamicSmemBytes = smem; cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = (unsigned)cluster; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        FIRE_CUDA_TRY(L, cudaLaunchKernelEx(&cfg, kernel, prm));
    } else {
        kernel<<<grid, threads, smem, st>>>(prm);
    }
    FIRE_CUDA_TRY(L, cudaGetLastError());
    if (prof) { FIRE_CUDA_TRY(L, cudaEventRecord(L->prof_ev[2 * L->prof_count + 1], st)); L->prof_count += 1; }
    {
        const size_t n = (size_t)L->Th * L->Ww;
        const dim3 fgrid((unsigned)((n + 255) / 256), (unsigned)(S < 65535 ? S : 65535));
        if (L->fit_counts) fire_finish_kernel<true><<<fgrid, 256, 0, st>>>(L->burnable, L->tiles, L->status + S, planes, out_burned, L->H, L->Ww, L->Tw, L->Th, S, L->fit_ref, L->fit_counts);
        else fire_finish_kernel<false><<<fgrid, 256, 0, st>>>(L->burnable, L->tiles, L->status + S, planes, out_burned, L->H, L->Ww, L->Tw, L->Th, S, nullptr, nullptr);
        FIRE_CUDA_TRY(L, cudaGetLastError());
    }
    if (bt) fire_propagate_rescue_bt_kernel<<<kRescueCtas, 256, 0, st>>>(prm, L->rescue_planes);
    else fire_propagate_rescue_kernel<<<kRescueCtas, 256, 0, st>>>(prm, L->rescue_planes);
    FIRE_CUDA_TRY(L, cudaGetLastError());
    L->launches += 4;
    return FIRE_OK;
}
