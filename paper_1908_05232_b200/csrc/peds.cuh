// peds.cuh -- steps (B), (P), (O), (S) and the scalar tail (T) of include/floodped.h.
//
// Pedestrians are stored SoA and re-sorted by bin every step (counting sort): this replaces
// FLAMEGPU's navigation-agent / spatially partitioned messages.  Bins are k x k
// flood cells with k dx >= R_int, so the 3 x 3 adjacent bins hold every interaction partner
// (C26); the three bins of one bin-row are contiguous in the sorted order, so the
// neighbourhood is three contiguous index ranges.
#pragma once

#include "common.cuh"

namespace fp {

template <typename T>
struct PedSoA {
    T *x, *y, *vx, *vy, *vpref, *timer;
    uint8_t *role, *fsm, *state, *active;
    int32_t *id;
    int32_t *cell;                   // level-n containing cell (valid in the sorted buffer)
};

// Where the flood state of a cell lives: row slab r = row / rows holds the rows
// [r rows, (r + 1) rows); every pointer is pre-offset so that it is indexed with the GLOBAL cell
// index.  One slab = the handle's own grid.  With several, the other slabs' arrays are peer memory
// (NVLink) or other handles on the same device.
constexpr int MAX_SLABS = 8;
template <typename T>
struct SlabTab {
    int n, rows;
    const T *h[2][MAX_SLABS], *qx[2][MAX_SLABS], *qy[2][MAX_SLABS];   // [flood parity][slab]
    uint8_t *occ[2][MAX_SLABS];                                          // [N_p buffer][slab]
    __device__ __forceinline__ int of(int c, int nx) const { return n == 1 ? 0 : min((c / nx) / rows, n - 1); }
};

template <typename T>
struct PedArgs {
    int n;                           // all agents, active or not
    int nx, ny, kbin, nbx, nby, nbins;
    T inv_dx, inv_dy, dxk;
    T h_dry, hr_edge[3], speed_wet[4];
    T inv_tau, A_s, inv_B, two_r, R_int, R2, vmax_factor, t_pick, t_drop;
    int n_targets, exit_target, storage_target, drop_target;
    int n_exit; int exit_i[16], exit_j[16];
    int storage_i, storage_j, drop_i, drop_j, arrive;
    int n_doors; int door_i[16], door_j[16], door_target[16];   // entrance doors: fsm = FSM_WANDER + destination door
    PedSoA<T> A, B;                  // A: level n (any order) and level n+1; B: level n sorted by bin
    VecN<T, 2> *bxy;                 // (x, y) of B interleaved: one 64/128-bit load per candidate
    T c_exp1, c_exp2;                // fp32 pair force: A_s e^{(2r-d)/B_s} = 2^{c_exp1 + c_exp2 d}
    int32_t *key, *off;              // per slot of A: bin key, rank inside the bin
    int32_t *perm;                   // deterministic mode only: [n] sorted slot -> slot of A (ped_perm_kernel)
    int32_t *count;                  // [nbins+1] (zeroed by the scan after use)
    int32_t *start;                  // [nbins+2] exclusive scan
    // N_p per cell is double-buffered by flood parity: the binning chain of step n+1 runs beside the
    // flood step n, which is still reading the N_p of step n (buffer ctl->parity)
    int32_t *cellprev;               // [2][n] per slot: cell whose occupancy this slot set the last time this buffer was filled, or -1
    size_t cellprev_stride;
    int occ_in_scatter;              // 1 (small crowds): the scatter kernel counts N_p itself, no ped_occ_kernel launch
    int pdl_early;                   // 1: let the next kernel of the chain be scheduled at once (large crowds), see pdl_trigger()
    int pipelined;                   // 1: fill buffer ctl->occ_next (published by the pedestrian step of the step before); 0: ctl->parity
    const uint8_t *mask;             // [ncell] 1 = solid
    const uint8_t *nav;              // [n_targets][ncell]
    SlabTab<T> slab;                 // flood state (level n is [ctl->parity]) and N_p of every cell
    Ctl *ctl;
};

constexpr int FSM_WANDER = 8;        // include/floodped.h SIM_FSM_WANDER

// Which N_p buffer a kernel of the binning chain fills, or -1 if the chain must not run.
// Pipelined (beside the tail kernel of the step before, which is rewriting parity and halt):
// the decision was taken by the pedestrian step before it; otherwise the control block is stable.
template <typename T> __device__ __forceinline__ int chain_sel(const PedArgs<T> &a)
{
    return a.pipelined ? a.ctl->occ_next : (a.ctl->halt ? -1 : a.ctl->parity);
}

template <typename T> __device__ __forceinline__ int cell_of(T x, T inv, int n)
{
    int i = (int)floor(mul_rn(x, inv));
    return min(max(i, 0), n - 1);
}

// ---------------------------------------------------------------------------------- (B) count
// Key of every agent and its rank inside the bin.  Agents arrive nearly sorted (last step's
// order), so lanes of a warp mostly share a key: one atomic per distinct key per warp
// (warp-aggregated atomics via match.any).  Also clears the occupancy set by the previous step.
template <typename T>
__device__ __forceinline__ void bin_count_one(const PedArgs<T> &a, const int s, const int sel, const int clear_occ)
{
    const unsigned lanes = __activemask();
    int key = a.nbins, cell = -1;
    if (a.A.active[s]) {
        const int ix = cell_of(a.A.x[s], a.inv_dx, a.nx), iy = cell_of(a.A.y[s], a.inv_dy, a.ny);
        cell = iy * a.nx + ix;
        key = (iy / a.kbin) * a.nbx + ix / a.kbin;
    }
    const unsigned peers = __match_any_sync(lanes, key);
    const int lane = threadIdx.x & 31, leader = __ffs(peers) - 1;
    int base = 0;
    if (lane == leader) base = atomicAdd(&a.count[key], __popc(peers));
    base = __shfl_sync(peers, base, leader);
    a.key[s] = key;
    a.off[s] = base + __popc(peers & ((1u << lane) - 1u));
    a.A.cell[s] = cell;
    if (clear_occ) {
        const int c = a.cellprev[sel * a.cellprev_stride + s];
        if (c >= 0) a.slab.occ[sel][a.slab.of(c, a.nx)][c] = 0;      // sparse clear: only cells that were set (no dense memset)
    }
}

template <typename T>
__global__ void __launch_bounds__(256) ped_bin_count_kernel(PedArgs<T> a, int clear_occ)
{
    if (a.pdl_early) pdl_trigger();
    pdl_wait();
    const int sel = chain_sel(a);
    if (sel < 0) return;
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= a.n) return;
    bin_count_one(a, s, sel, clear_occ);
}

// ---------------------------------------------------------------------------------- (B) scan
// Single-pass exclusive scan with decoupled look-back over tiles of SCAN_TILE counts.
// status word = (epoch*4 + flag) << 32 | value; flag 1 = tile aggregate, 2 = inclusive prefix.
// The epoch (one per executed step) makes stale flags of earlier steps read as "not ready", so
// the status array never needs clearing.  Also zeroes count[] for the next step and writes
// start[n_items] = total.
constexpr int SCAN_THREADS = 512, SCAN_ITEMS = 16, SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;   // 8192 counts per tile: 128-bit accesses, short look-back chain

__global__ void __launch_bounds__(SCAN_THREADS) scan_bins_kernel(int32_t *count, int32_t *start, int n_items,
                                                                 unsigned long long *status, Ctl *ctl, int pipelined, int pdl_early)
{
    __shared__ int warp_sum[SCAN_THREADS / 32];
    __shared__ int tile_s, excl_s;
    if (pdl_early) pdl_trigger();
    pdl_wait();
    if (pipelined ? ctl->occ_next < 0 : ctl->halt != 0) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) tile_s = (int)atomicAdd(&ctl->scan_ticket, 1u);
    __syncthreads();
    const int tile = tile_s;
    const unsigned epoch = ctl->scan_epoch;
    const int base = tile * SCAN_TILE + tid * SCAN_ITEMS;
    int v[SCAN_ITEMS], sum = 0;
    const bool full = base + SCAN_ITEMS <= n_items;    // all my items exist: 128-bit accesses
    if (full) {
        int4 *c4 = reinterpret_cast<int4 *>(count + base);
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS / 4; ++k) {
            const int4 q = c4[k];
            v[4 * k] = q.x; v[4 * k + 1] = q.y; v[4 * k + 2] = q.z; v[4 * k + 3] = q.w;
            c4[k] = make_int4(0, 0, 0, 0);
        }
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) sum += v[k];
    } else {
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) {
            const int i = base + k;
            v[k] = i < n_items ? count[i] : 0;
            if (i < n_items) count[i] = 0;
            sum += v[k];
        }
    }
    int inc = sum;                                    // inclusive scan of thread sums in the warp
    for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
    if (lane == 31) warp_sum[warp] = inc;
    __syncthreads();
    int warp_off = 0, tile_total = 0;
#pragma unroll
    for (int w = 0; w < SCAN_THREADS / 32; ++w) { const int ws = warp_sum[w]; if (w < warp) warp_off += ws; tile_total += ws; }
    // publish the aggregate, then look back (warp 0)
    if (warp == 0) {
        const unsigned long long tag = (unsigned long long)(epoch * 4u);
        if (lane == 0) {
            const unsigned long long w = ((tag + (tile == 0 ? 2ull : 1ull)) << 32) | (unsigned)tile_total;
            atomicExch(&status[tile], w);
        }
        int excl = 0;
        if (tile > 0) {
            int look = tile - 1;
            while (true) {
                const int idx = look - lane;
                unsigned long long w = 0; unsigned flag = 0;
                do {
                    if (idx >= 0) {
                        w = *((volatile unsigned long long *)&status[idx]);
                        const unsigned hi = (unsigned)(w >> 32);
                        flag = (hi >> 2) == epoch ? (hi & 3u) : 0u;
                    } else flag = 2u, w = 0;          // before tile 0: prefix 0
                } while (__any_sync(0xffffffffu, flag == 0u));
                const unsigned done = __ballot_sync(0xffffffffu, flag == 2u);
                const int first_done = done ? __ffs(done) - 1 : 32;
                int val = lane <= first_done ? (int)(unsigned)(w & 0xffffffffull) : 0;
                for (int o = 16; o > 0; o >>= 1) val += __shfl_xor_sync(0xffffffffu, val, o);
                excl += val;
                if (done) break;
                look -= 32;
            }
            if (lane == 0) {
                const unsigned long long w = ((tag + 2ull) << 32) | (unsigned)(excl + tile_total);
                atomicExch(&status[tile], w);
            }
        }
        if (lane == 0) excl_s = excl;
    }
    __syncthreads();
    int run = excl_s + warp_off + (inc - sum);
    if (full) {
        int4 *s4 = reinterpret_cast<int4 *>(start + base);
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS / 4; ++k) {
            int4 q;
            q.x = run; run += v[4 * k];
            q.y = run; run += v[4 * k + 1];
            q.z = run; run += v[4 * k + 2];
            q.w = run; run += v[4 * k + 3];
            s4[k] = q;
        }
        if (base + SCAN_ITEMS == n_items) start[n_items] = run;
    } else {
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) {
            const int i = base + k;
            if (i < n_items) start[i] = run;
            run += v[k];
            if (i == n_items - 1) start[n_items] = run;
        }
    }
}

// ---------------------------------------------------------------------------------- (B) order
// Deterministic mode (sim_set_deterministic).  The rank an agent takes inside its bin above is the
// return value of an atomicAdd, i.e. the order in which warps happened to arrive: the sorted buffer
// is a valid counting sort, but which slot of its bin an agent lands in differs from run to run,
// and the pair loop sums the forces in slot order, so the last bits of every agent in a
// crowd differ too.  These two kernels, run between the scan and the scatter, replace that rank by
// the agent's rank BY ORIGINAL ID among the agents of its bin: the sorted order becomes a pure
// function of the (id, position) set -- the same on every run, for any number of row slabs and
// whatever order the agents were handed over in -- and it is the order in which the oracle walks
// its cell lists (increasing agent index per bin).
//   ped_perm_kernel : perm[start[key] + atomic rank] = slot of A  (which agents share a bin)
//   ped_rank_kernel : one thread per sorted slot counts the ids of its bin below its own: O(k) per
//                     agent, k = agents per bin (a handful on Configs 1-4, about 30 on Config 5).
// The slots past the last bin (inactive agents, key = nbins) keep their arrival order: nothing but
// the order output of sim_bin_peds reads them by slot, and there may be 10^6 of them.
template <typename T>
__global__ void __launch_bounds__(256) ped_perm_kernel(PedArgs<T> a)
{
    if (a.pdl_early) pdl_trigger();
    pdl_wait();
    if (chain_sel(a) < 0) return;
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= a.n) return;
    a.perm[a.start[a.key[s]] + a.off[s]] = s;
}

template <typename T>
__global__ void __launch_bounds__(256) ped_rank_kernel(PedArgs<T> a)
{
    if (a.pdl_early) pdl_trigger();
    pdl_wait();
    if (chain_sel(a) < 0) return;
    const int d = blockIdx.x * blockDim.x + threadIdx.x;
    if (d >= a.n) return;
    const int s = a.perm[d], b = a.key[s];
    if (b >= a.nbins) return;
    const int id = a.A.id[s];
    int below = 0;
    for (int j = a.start[b]; j < a.start[b + 1]; ++j) below += a.A.id[a.perm[j]] < id;
    a.off[s] = below;
}

// ---------------------------------------------------------------------------------- (B) scatter
template <typename T>
__global__ void __launch_bounds__(256) ped_scatter_kernel(PedArgs<T> a)
{
    if (a.pdl_early) pdl_trigger();
    pdl_wait();
    if (chain_sel(a) < 0) return;
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= a.n) return;
    if (s == 0) { a.ctl->scan_ticket = 0u; a.ctl->scan_epoch += 1u; }   // the scan before me is done: re-arm it for the next chain
    const int d = a.start[a.key[s]] + a.off[s];
    const T x = a.A.x[s], y = a.A.y[s];
    a.B.x[d] = x; a.B.y[d] = y; a.bxy[d] = VecN<T, 2>{x, y};
    a.B.vx[d] = a.A.vx[s]; a.B.vy[d] = a.A.vy[s];
    a.B.vpref[d] = a.A.vpref[s]; a.B.timer[d] = a.A.timer[s];
    a.B.role[d] = a.A.role[s]; a.B.fsm[d] = a.A.fsm[s]; a.B.state[d] = a.A.state[s];
    a.B.active[d] = a.A.active[s]; a.B.id[d] = a.A.id[s]; a.B.cell[d] = a.A.cell[s];
    // small crowds: N_p per cell here, one launch fewer on the critical path of the step.
    // Saturating add of 1 to the cell's byte by compare-and-swap on its word (the cells that were set
    // the last time this buffer was filled have been cleared by the count kernel before).
    if (a.occ_in_scatter) {
        const int sel = chain_sel(a);
        int32_t *cellprev = a.cellprev + sel * a.cellprev_stride;
        if (!a.A.active[s]) { cellprev[d] = -1; return; }
        const int c = a.A.cell[s];
        uint8_t *p = a.slab.occ[sel][a.slab.of(c, a.nx)] + c;
        unsigned int *w = reinterpret_cast<unsigned int *>(reinterpret_cast<uintptr_t>(p) & ~uintptr_t(3));
        const int sh = 8 * (int)(reinterpret_cast<uintptr_t>(p) & 3);
        unsigned int old = *w;
        while (((old >> sh) & 255u) != 255u) {
            const unsigned int seen = atomicCAS(w, old, old + (1u << sh));
            if (seen == old) break;
            old = seen;
        }
        cellprev[d] = c;
    }
}

// ---------------------------------------------------------------------------------- (O)
// N_p per cell from the sorted level-n agents: the agents of a cell all sit in one bin, so
// each agent counts those of its own bin that share its cell and the lowest slot publishes the
// count.  Also remembers the cell so that next step's bin count can clear it (sparse clear).
// Runs before the flood kernel, which consumes occ[]; the pedestrian step itself does not need it.
template <typename T>
__global__ void __launch_bounds__(256) ped_occ_kernel(PedArgs<T> a)
{
    if (a.pdl_early) pdl_trigger();
    pdl_wait();
    const int sel = chain_sel(a);
    if (sel < 0) return;
    const int d = blockIdx.x * blockDim.x + threadIdx.x;
    if (d >= a.n) return;
    int32_t *cellprev = a.cellprev + sel * a.cellprev_stride;
    if (!a.B.active[d]) { cellprev[d] = -1; return; }
    const int c = a.B.cell[d];
    const int b = ((c / a.nx) / a.kbin) * a.nbx + (c % a.nx) / a.kbin;
    int same = 0, lower = 0;
    for (int j = a.start[b]; j < a.start[b + 1]; ++j)
        if (a.B.cell[j] == c) { same += 1; lower += (j < d); }
    if (lower == 0) a.slab.occ[sel][a.slab.of(c, a.nx)][c] = (uint8_t)min(same, 255);
    cellprev[d] = c;
}

// ---------------------------------------------------------------------------------- (P) pair loop
// One candidate of the pair loop: adds A_s exp((2r - d)/B_s) (x_i - x_j)/d to (ax, ay) if 0 < d < R_int
// (C24, C26).
//   fp32: the difference and its squares on packed FADD2 / FFMA2; the squares carry +5e-31 each, so
//   d2 >= 1e-30 > 0 and the agent itself or a coincident partner (d = 0, skipped by C26) needs no
//   second compare: its force factor is finite and multiplies dx = dy = 0.  Two MUFU (rsqrt, ex2);
//   the force constants are read from memory once per thread (Ctl::pair_c1).  12 instructions per
//   candidate (16 in round 1).  The kernel stays bound by the XU pipe: a predicated-off MUFU still
//   occupies it for the whole warp, and two thirds of the candidates of the 3 x 3 bins lie outside
//   R_int.  Three ways of issuing the MUFU pair only for pairs inside the cut-off were built and
//   measured on Config 5: all of them cost more issue slots than the XU cycles they save.
template <typename T> struct PairConst { T R2, c1, c2; };
template <typename T> __device__ __forceinline__ PairConst<T> pair_const(const PedArgs<T> &a)
{
    PairConst<T> k{a.R2, a.c_exp1, a.c_exp2};
    if constexpr (sizeof(T) == 4) { k.c1 = a.ctl->pair_c1; k.c2 = a.ctl->pair_c2; }   // see Ctl
    return k;
}

__device__ __forceinline__ void pair_add(const PedArgs<float> &, const PairConst<float> &k, float x, float y, VecN<float, 2> pj, float &ax, float &ay)
{
    const f2 dd = sub2(pk(x, y), pk(pj.v[0], pj.v[1]));
    const f2 sq = fma2(dd, dd, pk1(5e-31f));
    const float d2 = sq.x + sq.y;
    if (d2 < k.R2) {
        const float rinv = fast_rsqrt(d2);
        float e;
        asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(fmaf(d2 * rinv, k.c2, k.c1)));
        const float f = e * rinv;
        ax = fmaf(f, dd.x, ax); ay = fmaf(f, dd.y, ay);
    }
}
__device__ __forceinline__ void pair_add(const PedArgs<double> &a, const PairConst<double> &, double x, double y, VecN<double, 2> pj, double &ax, double &ay)
{
    const double ddx = x - pj.v[0], ddy = y - pj.v[1];
    const double d2 = ddx * ddx + ddy * ddy;
    if (d2 > 0.0 && d2 < a.R2) {
        const double d = sqrt(d2);
        const double f = a.A_s * exp((a.two_r - d) * a.inv_B) / d;
        ax += f * ddx; ay += f * ddy;
    }
}

#ifndef PED_UNROLL
#define PED_UNROLL 8
#endif
#ifndef PED_THREADS_N
#define PED_THREADS_N 128
#endif
constexpr int PED_THREADS = PED_THREADS_N;
constexpr int PED_UNROLL_K = PED_UNROLL;

// ---------------------------------------------------------------------------------- (P)+(O)
// One thread per sorted slot d: reads level n from B (+ flood level n), writes level n+1 to A[d].
// Independent of the flood kernel of the same step (both read level n), so the two may overlap.
template <typename T>
__device__ __forceinline__ void ped_step_one(const PedArgs<T> &a, const int d)
{
    const PedSoA<T> &B = a.B, &A = a.A;
    const T x = B.x[d], y = B.y[d], vx = B.vx[d], vy = B.vy[d], vpref = B.vpref[d];
    T timer = B.timer[d];
    const uint8_t role = B.role[d], act = B.active[d];
    uint8_t fsm = B.fsm[d], state = B.state[d];
    const int c = B.cell[d];
    A.vpref[d] = vpref; A.role[d] = role; A.id[d] = B.id[d];
    if (!act) {
        A.x[d] = x; A.y[d] = y; A.vx[d] = vx; A.vy[d] = vy; A.timer[d] = timer;
        A.fsm[d] = fsm; A.state[d] = state; A.active[d] = 0;
        return;
    }
    const int ix = c % a.nx, iy = c / a.nx;
    const int bx = ix / a.kbin, by = iy / a.kbin;

    // 4. social repulsion over the 3 x 3 adjacent bins (C24, C26): three contiguous
    //    index ranges, one per bin row
    T ax = T(0), ay = T(0);
    const PairConst<T> kc = pair_const(a);
    for (int jy = max(by - 1, 0); jy <= min(by + 1, a.nby - 1); ++jy) {
        const int s0 = a.start[jy * a.nbx + max(bx - 1, 0)];
        const int s1 = a.start[jy * a.nbx + min(bx + 1, a.nbx - 1) + 1];
#pragma unroll PED_UNROLL_K
        for (int j = s0; j < s1; ++j) pair_add(a, kc, x, y, a.bxy[j], ax, ay);
    }
    // D7: once water is in the domain those still wandering become evacuees;
    // D6: before that a wanderer leaves through its destination door, not through the exit
    bool out = false;
    if (fsm >= FSM_WANDER) {
        if (a.ctl->triggered) fsm = 0;
        else out = max(abs(ix - a.door_i[fsm - FSM_WANDER]), abs(iy - a.door_j[fsm - FSM_WANDER])) <= a.arrive;
    }
    // 8. exit (C29): level-n cell within arrive_cells of an exit cell
    if (fsm < FSM_WANDER && (role == 0 || fsm == 0))
        for (int e = 0; e < a.n_exit; ++e)
            out |= max(abs(ix - a.exit_i[e]), abs(iy - a.exit_j[e])) <= a.arrive;
    if (out) {
        A.x[d] = x; A.y[d] = y; A.vx[d] = vx; A.vy[d] = vy; A.timer[d] = timer;
        A.fsm[d] = fsm; A.state[d] = state; A.active[d] = 0;
        return;
    }
    // 1. sample U^n at the containing cell -> HR -> Table 1 (C17-C20)
    const int p = a.ctl->parity;
    const int sl = a.slab.of(c, a.nx);
    const T h = a.slab.h[p][sl][c];
    T u = T(0), v = T(0);
    if (h > a.h_dry) { u = div_rn(a.slab.qx[p][sl][c], h); v = div_rn(a.slab.qy[p][sl][c], h); }
    const T hr = mul_rn(add_rn(fmax(fabs(u), fabs(v)), T(0.5)), h);
    if (!(h > a.h_dry)) state = 0;
    else if (hr < a.hr_edge[0]) state = 1;
    else if (hr < a.hr_edge[1]) state = 2;
    else if (hr < a.hr_edge[2]) state = 3;
    else state = 4;
    // 2. desired speed
    T v0 = state == 0 ? vpref : a.speed_wet[state - 1];
    if (fsm == 2 || fsm == 4) v0 = T(0);
    // 3. desired direction from the navigation field of the current target
    int target = a.exit_target;
    if (fsm == 1) target = a.storage_target; else if (fsm == 3) target = a.drop_target;
    else if (fsm >= FSM_WANDER) target = a.door_target[fsm - FSM_WANDER];
    const int code = a.nav[(size_t)target * ((size_t)a.nx * a.ny) + c];
    T ex = T(0), ey = T(0);
    if (code < 8) {
        const T r = T(0.70710678118654752440);
        const int dxs = (code == 0 || code == 1 || code == 7) - (code == 3 || code == 4 || code == 5);
        const int dys = (code == 1 || code == 2 || code == 3) - (code == 5 || code == 6 || code == 7);
        const T m = (dxs != 0 && dys != 0) ? r : T(1);
        ex = m * T(dxs); ey = m * T(dys);
    }
    // 5. velocity: backward Euler on the relaxation term (C25), speed cap
    const T dt = (T)a.ctl->dt;
    const T den = T(1) / (T(1) + dt * a.inv_tau);
    T wx = (vx + dt * (v0 * ex * a.inv_tau + ax)) * den;
    T wy = (vy + dt * (v0 * ey * a.inv_tau + ay)) * den;
    const T wmax = a.vmax_factor * v0, wn = real_sqrt(wx * wx + wy * wy);
    if (wn > wmax) { const T f = wn > T(0) ? wmax / wn : T(0); wx *= f; wy *= f; }
    // 6. move, axis by axis, rejecting moves into solids or out of the domain (C27)
    auto blocked = [&](T px, T py) {
        const T fi = floor(mul_rn(px, a.inv_dx)), fj = floor(mul_rn(py, a.inv_dy));
        if (fi < T(0) || fi >= T(a.nx) || fj < T(0) || fj >= T(a.ny)) return true;
        return a.mask[(int)fj * a.nx + (int)fi] != 0;
    };
    T xn = x + dt * wx, yn = y;
    if (blocked(xn, yn)) { xn = x; wx = T(0); }
    yn = y + dt * wy;
    if (blocked(xn, yn)) { yn = y; wy = T(0); }
    // 7. responder FSM on the level-n cell (C31)
    if (role == 1) {
        if (fsm == 1) {
            if (max(abs(ix - a.storage_i), abs(iy - a.storage_j)) <= a.arrive) { fsm = 2; timer = a.t_pick; }
        } else if (fsm == 2) {
            timer = add_rn(timer, -dt);
            if (timer <= T(0)) fsm = 3;
        } else if (fsm == 3) {
            if (max(abs(ix - a.drop_i), abs(iy - a.drop_j)) <= a.arrive) { fsm = 4; timer = a.t_drop; }
        } else if (fsm == 4) {
            timer = add_rn(timer, -dt);
            if (timer <= T(0)) { atomicAdd(&a.ctl->D, 1); fsm = a.ctl->complete ? 0 : 1; }
        }
    }
    A.x[d] = xn; A.y[d] = yn; A.vx[d] = wx; A.vy[d] = wy; A.timer[d] = timer;
    A.fsm[d] = fsm; A.state[d] = state; A.active[d] = 1;
}


// fuse_count = 1 (step graph): every thread goes on to key and count its own agent for the binning
// chain of the NEXT step (the first kernel of that chain folded in: one launch fewer on the
// critical path of small crowds).  The chain fills N_p buffer parity ^ 1, which the flood kernel
// running beside this one does not read.
template <typename T>
__global__ void __launch_bounds__(PED_THREADS) ped_step_kernel(PedArgs<T> a, int fuse_count)
{
    pdl_enter();
    const int d = blockIdx.x * blockDim.x + threadIdx.x;
    const int halt = a.ctl->halt, sel = a.ctl->parity ^ 1;
    // for the binning chain of the next step, which runs beside this step's tail kernel: go / no go
    if (d == 0) a.ctl->occ_next = halt ? -1 : sel;
    if (halt) return;
    if (d >= a.n) return;
    ped_step_one(a, d);
    if (fuse_count) bin_count_one(a, d, sel, 1);
}

// ---------------------------------------------------------------------------------- (S)+(T) tail
// One thread: sandbag arithmetic, time, next dt, next inflow.
template <typename T>
struct TailArgs {
    Ctl *ctl;
    T *zs_tab[MAX_SLABS];            // bed of every row slab, pre-offset for the global cell index (8f-4)
    int slab_rows, nx, n_slabs;
    const int32_t *line_cells;
    int n_line, bags_per_cell_layer, n_layers;
    T layer_thickness;
    const double *hydro_t, *hydro_q;
    int n_hydro;
    double inv_inflow_length;
    // entrance doors
    PedSoA<T> A;                     // level n+1 pedestrians (after the pedestrian step of this step)
    int np, n_doors;
    int door_cells[16];
    double *door_credit;             // [16] newcomers owed by each door
    double spawn_rate, vpref_lo, vpref_hi, dx, dy;
    int target_population;
    unsigned int seed_lo, seed_hi;
};

// Philox4x32-10 (Salmon et al., SC'11) written from its definition; known answers: tests/test_boundary.py
__device__ __forceinline__ void philox4x32_10(unsigned c0, unsigned c1, unsigned c2, unsigned c3, unsigned k0, unsigned k1, unsigned out[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        const unsigned h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ k0; c1 = l1; c2 = h0 ^ c3 ^ k1; c3 = l0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

__global__ void philox_test_kernel(const unsigned *in /* [n][6] */, unsigned *out /* [n][4] */, int n)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) philox4x32_10(in[6 * k], in[6 * k + 1], in[6 * k + 2], in[6 * k + 3], in[6 * k + 4], in[6 * k + 5], out + 4 * k);
}

// D3-D5: the doors let newcomers in.  One warp; every lane holds the same copy of the control block.
// The free-slot search (lowest original index among the inactive slots, D4) and the head count
// are strided scans over the level n+1 arrays with a warp reduction: once per newcomer, which is a
// few per step at most (10 per door).
template <typename T>
__device__ __forceinline__ void spawn_warp(const TailArgs<T> &a, long long &spawned, const double dt_taken)
{
    const int lane = threadIdx.x & 31;
    const volatile uint8_t *act = a.A.active;
    int pop = 0;
    for (int s = lane; s < a.np; s += 32) pop += act[s] ? 1 : 0;
    pop = __reduce_add_sync(0xffffffffu, pop);
    for (int d = 0; d < a.n_doors; ++d) {
        double cr = __dadd_rn(a.door_credit[d], __dmul_rn(a.spawn_rate, dt_taken));
        while (cr >= 1.0) {
            unsigned long long best = ~0ull;
            if (pop < a.target_population)
                for (int s = lane; s < a.np; s += 32)
                    if (!act[s]) { const unsigned long long k = ((unsigned long long)(unsigned)a.A.id[s] << 32) | (unsigned)s; best = k < best ? k : best; }
            for (int o = 16; o > 0; o >>= 1) { const unsigned long long t = __shfl_xor_sync(0xffffffffu, best, o); best = t < best ? t : best; }
            if (best == ~0ull) { cr = 1.0; break; }                     // full: the door waits, owing one
            if (lane == 0) {
                const int s = (int)(unsigned)(best & 0xffffffffull);
                unsigned r[4];
                philox4x32_10((unsigned)(spawned & 0xffffffffll), (unsigned)(spawned >> 32), 0u, 0u, a.seed_lo, a.seed_hi, r);
                const int dest = (int)(((unsigned long long)r[0] * (unsigned long long)a.n_doors) >> 32);
                const double k32 = 1.0 / 4294967296.0;
                const double ux = __dmul_rn((double)r[1], k32), uy = __dmul_rn((double)r[2], k32), uv = __dmul_rn((double)r[3], k32);
                const int ci = a.door_cells[d] % a.nx, cj = a.door_cells[d] / a.nx;
                a.A.x[s] = (T)__dmul_rn(__dadd_rn(__dadd_rn((double)ci, 0.1), __dmul_rn(0.8, ux)), a.dx);
                a.A.y[s] = (T)__dmul_rn(__dadd_rn(__dadd_rn((double)cj, 0.1), __dmul_rn(0.8, uy)), a.dy);
                a.A.vx[s] = T(0); a.A.vy[s] = T(0); a.A.timer[s] = T(0);
                a.A.vpref[s] = (T)__dadd_rn(a.vpref_lo, __dmul_rn(__dadd_rn(a.vpref_hi, -a.vpref_lo), uv));
                a.A.role[s] = 0; a.A.state[s] = 0; a.A.fsm[s] = (uint8_t)(FSM_WANDER + dest);
                a.A.active[s] = 1;
                __threadfence();
            }
            __syncwarp();
            cr = __dadd_rn(cr, -1.0); spawned += 1; pop += 1;
        }
        if (lane == 0) a.door_credit[d] = cr;
    }
}

__device__ __forceinline__ double hydrograph(const double *t, const double *q, int n, double time)
{
    if (n <= 0) return 0.0;
    if (time <= t[0]) return q[0];
    for (int k = 0; k + 1 < n; ++k)
        if (time < t[k + 1]) return q[k] + (q[k + 1] - q[k]) * (time - t[k]) / (t[k + 1] - t[k]);
    return q[n - 1];
}

// hydrograph() with the table spread over the lanes of a warp: all entries are loaded at once
// (one memory latency instead of one per segment -- this kernel sits on the critical path of every
// step).  Same segments, same interpolation expression.  All 32 lanes must call it.
__device__ __forceinline__ double hydrograph_warp(const double *t, const double *q, int n, double time)
{
    if (n <= 0) return 0.0;
    const int lane = threadIdx.x & 31;
    double res = 0.0;
    bool found = false;
    if (time <= t[0]) { res = q[0]; found = true; }            // warp-uniform
    for (int base = 0; base + 1 < n && !found; base += 32) {
        const int k = base + lane;
        const bool ok = k + 1 < n;
        const double t0 = ok ? t[k] : 0.0, t1 = ok ? t[k + 1] : 0.0, q0 = ok ? q[k] : 0.0, q1 = ok ? q[k + 1] : 0.0;
        const unsigned hit = __ballot_sync(0xffffffffu, ok && time < t1);
        if (hit) {
            const int src = __ffs(hit) - 1;
            const double v = q0 + (q1 - q0) * (time - t0) / (t1 - t0);
            res = __shfl_sync(0xffffffffu, v, src);
            found = true;
        }
    }
    if (!found) res = q[n - 1];
    return res;
}

// first = 1: only derive dt and q_in from the state already in place (create / test hooks).
// One warp; lane 0 owns the control block.  It works on a register copy read with independent
// loads and writes back only the fields this kernel owns: the binning chain of the next step may
// be running beside it and owns scan_ticket / scan_epoch / occ_next.
template <typename T>
__global__ void tail_kernel(TailArgs<T> a, int first)
{
    pdl_enter();
    if (blockIdx.x != 0 || threadIdx.x >= 32) return;
    Ctl *c = a.ctl;
    Ctl l = *c;
    if (!first && l.halt) return;                              // warp-uniform
    if (!first) {
        if (threadIdx.x == 0 && l.D > 0) {                     // deposits of this step
            const int D = l.D;
            l.deposits += D;
            for (int d = 0; d < D && !l.complete; ++d) {
                l.bags += 1;
                if (l.bags == a.bags_per_cell_layer) {
                    const int lc = a.line_cells[l.cursor];
                    a.zs_tab[min(lc / a.nx / a.slab_rows, a.n_slabs - 1)][lc] += a.layer_thickness;   // as SlabTab::of: the last slab may be the longer one
                    l.bags = 0; l.cursor += 1;
                    if (l.cursor == a.n_line) { l.layer += 1; l.cursor = 0; }
                    if (l.layer == a.n_layers) l.complete = 1;
                }
            }
            c->deposits = l.deposits; c->bags = l.bags; c->cursor = l.cursor; c->layer = l.layer; c->complete = l.complete;
        }
        l.t += l.dt;
        l.step += 1;
        l.parity ^= 1;
    }
    const double lam = __longlong_as_double((long long)l.lam_bits);
    // D7, D8: a wet cell exists in U^{n+1} (its wave speed is positive) -> triggered, for good;
    // D3: otherwise the doors let newcomers in (they exist from level n+1 on)
    if (lam > 0.0) l.triggered = 1;
    if (!first && !l.triggered && a.n_doors > 0) spawn_warp(a, l.spawned, l.dt);
    double dt = l.dt_max;
    if (lam > 0.0) dt = fmin(dt, l.cfl / lam);
    if (l.t + dt > l.t_end) dt = fmax(0.0, l.t_end - l.t);
    const double q_in = hydrograph_warp(a.hydro_t, a.hydro_q, a.n_hydro, l.t) * a.inv_inflow_length;
    if (threadIdx.x == 0) {
        if (!first) { c->D = 0; c->t = l.t; c->step = l.step; c->parity = l.parity; }
        c->dt = dt;
        c->triggered = l.triggered; c->spawned = l.spawned;
        c->lam_bits = 0ull;
        c->halt = (l.t >= l.t_end) ? 1 : 0;
        c->q_in = q_in;
    }
}

// Row slabs: the global time step is the minimum over the slabs, i.e. the
// maximum of their wave speeds: every slab's control block receives the maximum over all of them.
struct SlabCtls { Ctl *c[MAX_SLABS]; int n; };
__global__ void slab_lambda_kernel(SlabCtls t)
{
    if (blockIdx.x != 0 || threadIdx.x != 0) return;
    unsigned long long m = 0ull;
    for (int r = 0; r < t.n; ++r) { const unsigned long long v = t.c[r]->lam_bits; m = v > m ? v : m; }   // non-negative doubles order like integers
    for (int r = 0; r < t.n; ++r) t.c[r]->lam_bits = m;
}

// ---------------------------------------------------------------------------------- read-back
// un-permute to original index order ("coordinates and states of the pedestrian agents")
template <typename T>
__global__ void ped_gather_kernel(PedSoA<T> A, int n, int nx, T inv_dx, T inv_dy, int ny,
                                  T *x, T *y, T *vx, T *vy, uint8_t *state, uint8_t *fsm,
                                  uint8_t *active, int32_t *cell, T *timer, int32_t *order)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const int i = A.id[s];
    if (x) x[i] = A.x[s];
    if (y) y[i] = A.y[s];
    if (vx) vx[i] = A.vx[s];
    if (vy) vy[i] = A.vy[s];
    if (state) state[i] = A.state[s];
    if (fsm) fsm[i] = A.fsm[s];
    if (active) active[i] = A.active[s];
    if (cell) cell[i] = cell_of(A.y[s], inv_dy, ny) * nx + cell_of(A.x[s], inv_dx, nx);
    if (timer) timer[i] = A.timer[s];
    if (order) order[s] = i;
}

template <typename T>
__global__ void ped_key_by_id_kernel(PedSoA<T> A, const int32_t *key, int n, int32_t *key_by_id)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n) key_by_id[A.id[s]] = key[s];
}

// state histogram for sim_get_stats: hist[0..4] active by state, hist[5] = left the domain
template <typename T>
__global__ void __launch_bounds__(256) ped_hist_kernel(PedSoA<T> A, int n, unsigned long long *hist, double *n_bad)
{
    __shared__ unsigned int sh[7];                     // per-block counts: 6 classes + non-finite
    if (threadIdx.x < 7) sh[threadIdx.x] = 0u;
    __syncthreads();
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n) {
        const int k = A.active[s] ? min((int)A.state[s], 4) : 5;
        const unsigned peers = __match_any_sync(__activemask(), k);
        if ((threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(&sh[k], (unsigned)__popc(peers));
        if (!isfinite((double)A.x[s]) || !isfinite((double)A.y[s])) atomicAdd(&sh[6], 1u);
    }
    __syncthreads();
    if (threadIdx.x < 6 && sh[threadIdx.x]) atomicAdd(&hist[threadIdx.x], (unsigned long long)sh[threadIdx.x]);
    if (threadIdx.x == 6 && sh[6]) atomicAdd(n_bad, (double)sh[6]);
}

}  // namespace fp
