// floodped.cu -- the C ABI of include/floodped.h over the kernels in flood.cuh / peds.cuh.
// Host code only marshals, validates, places state in one device workspace and enqueues
// kernels (as CUDA graphs); every step of the path runs in the kernels.
#include "../../include/floodped.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <limits>
#include <mutex>
#include <cstdlib>
#include <string>
#include <vector>

#include "flood.cuh"
#include "flood_march.cuh"
#include "flood_march2.cuh"
#include "flood_tmarch.cuh"
#include "flood_muscl.cuh"
#include "peds.cuh"

using namespace fp;

namespace {

thread_local std::string g_create_error;

constexpr int GRAPH_LEVELS = 7;     // step graphs of 1, 2, 4, ... 64 coupled steps: any n is a few gap-free replays

struct Bump {                       // carve device state out of one workspace
    char *base = nullptr; size_t off = 0, cap = 0; bool dry = true;
    template <typename U> U *take(size_t n)
    {
        off = (off + 255) & ~size_t(255);
        U *p = dry ? nullptr : reinterpret_cast<U *>(base + off);
        off += n * sizeof(U);
        return p;
    }
};

}  // namespace

struct sim {
    sim_grid_t grid{};
    sim_params_t prm{};             // scalar copy; pointers inside are NOT valid after create
    int ncell = 0, np = 0, kbin = 1, nbx = 0, nby = 0, nbins = 0;
    // row slab: the flood arrays hold rows [j0, j0 + grid.ny) of a grid of gny rows; the
    // pedestrians (all of them live on the first slab's handle) walk on the whole grid of pcell cells
    int gny = 0, j0 = 0, pcell = 0;
    // linked slabs in row order (sim_slab_link: handles of this process; sim_slab_attach: raw device addresses,
    // e.g. of other processes' workspaces mapped through CUDA IPC)
    struct Peer { int j0 = 0, ny = 0; void *h[2]{}, *qx[2]{}, *qy[2]{}, *zs = nullptr; uint8_t *occ = nullptr; Ctl *ctl = nullptr; } peer[8];
    sim *group[8]{}; int ngroup = 0, grank = 0;
    cudaEvent_t ev_slab = nullptr;
    int n_inflow = 0, n_hydro = 0, n_line = 0, n_targets = 0;
    double inflow_length = 0.0;
    cudaStream_t stream = nullptr, cap_stream = nullptr;
    void *ws = nullptr; size_t ws_bytes = 0; bool own_ws = false;
    // device arrays (void*: real type decided by grid.real_bits)
    void *h[2]{}, *qx[2]{}, *qy[2]{}, *zs = nullptr, *z0 = nullptr, *n0 = nullptr, *scratch_real[3]{};
    uint8_t *occ = nullptr, *mask = nullptr, *inflow[4]{}, *nav = nullptr;
    int32_t *line_cells = nullptr;
    int line_row_max = -1;           // highest grid row that holds a barrier cell (host copy for sim_slab_attach)
    double *hydro_t = nullptr, *hydro_q = nullptr;
    struct { void *x, *y, *vx, *vy, *vpref, *timer; uint8_t *role, *fsm, *state, *active; int32_t *id, *cell; } P[2]{};
    void *ped_out[5]{};             // gather targets (x y vx vy timer) in original order
    uint8_t *ped_out_u8[3]{};
    int32_t *ped_out_i32[2]{};
    int32_t *key = nullptr, *off = nullptr, *count = nullptr, *start = nullptr, *cellprev = nullptr;
    int32_t *perm = nullptr; int deterministic = 0;       // sim_set_deterministic: bins ordered by original id
    void *bxy = nullptr;              // (x, y) of the sorted level-n agents, interleaved, for the pair loop
    unsigned long long *scan_status = nullptr;
    Ctl *ctl = nullptr;
    double *stat_d = nullptr;       // [4] volume, max_h, max_hr, n_bad ; [4] ped bad
    unsigned long long *stat_hist = nullptr;   // [6]
    int flood_variant = 1;
    int march_R = 64, march_gx = 1, march_gy = 1;
    uint8_t *chunk_flag = nullptr;
    uint8_t *dryseg = nullptr; size_t dry_stride = 0; int nsegx = 0; int dry_skip = 1;   // dry-segment flags of the TMA march kernel
    void *ghost_zero = nullptr, *ghost_inf = nullptr;   // one strip-wide row each (TMA kernel, rows beyond the domain)
    int exit_i[16]{}, exit_j[16]{};
    int door_cells[16]{}, door_target[16]{};
    double *door_credit = nullptr;             // [16] device
    cudaGraphExec_t graph[GRAPH_LEVELS]{};          // graph[k] advances 2^k coupled steps; built on first use
    int device = 0;                   // the device the handle lives on; every entry point runs on it
    int n_sm = 148;
    cudaStream_t stream2 = nullptr;   // second branch of the step graph (pedestrian step beside the flood step)
    cudaEvent_t ev_fork = nullptr, ev_ped = nullptr, ev_occ = nullptr, ev_tail = nullptr;
    int overlap = 1;
    int pdl = 1;                     // programmatic dependent launch inside the step graph
    bool binned = false;             // the binning chain of the upcoming step has run on the current state
    std::string err;
};

namespace {

int fail(sim *s, int code, const std::string &msg)
{
    if (s) s->err = msg; else g_create_error = msg;
    return code;
}

#define CU(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(s, SIM_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_));         \
    } while (0)

size_t real_size(const sim *s) { return s->grid.real_bits == 64 ? 8 : 4; }

// Every entry point runs on the device the handle was created on, whatever the caller's current
// device is, and leaves the caller's device as it found it.
struct DeviceGuard {
    int prev = -1; bool switched = false;
    explicit DeviceGuard(const sim *s)
    {
        if (s && cudaGetDevice(&prev) == cudaSuccess && prev != s->device) switched = cudaSetDevice(s->device) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

// Lay out (dry = true: only measure) all device state.
size_t layout(sim *s, Bump &b)
{
    const size_t rs = real_size(s), nc = (size_t)s->ncell, np = (size_t)s->np;
    auto real = [&](size_t n) { return (void *)b.take<char>(n * rs); };
    s->ctl = b.take<Ctl>(1);
    s->door_credit = b.take<double>(16);
    s->stat_d = b.take<double>(8);
    s->stat_hist = b.take<unsigned long long>(8);
    for (int k = 0; k < 2; ++k) { s->h[k] = real(nc); s->qx[k] = real(nc); s->qy[k] = real(nc); }
    s->zs = real(nc); s->z0 = real(nc); s->n0 = real(nc);
    for (int k = 0; k < 3; ++k) s->scratch_real[k] = real(nc);
    s->occ = b.take<uint8_t>(2 * nc); s->mask = b.take<uint8_t>((size_t)(s->np > 0 ? s->pcell : 1));
    s->inflow[0] = b.take<uint8_t>(s->grid.ny); s->inflow[1] = b.take<uint8_t>(s->grid.ny);
    s->inflow[2] = b.take<uint8_t>(s->grid.nx); s->inflow[3] = b.take<uint8_t>(s->grid.nx);
    s->nav = b.take<uint8_t>(s->np > 0 ? (size_t)s->n_targets * s->pcell : 1);
    s->line_cells = b.take<int32_t>(s->n_line + 1);
    s->hydro_t = b.take<double>(s->n_hydro + 1); s->hydro_q = b.take<double>(s->n_hydro + 1);
    for (int k = 0; k < 2; ++k) {
        s->P[k].x = real(np); s->P[k].y = real(np); s->P[k].vx = real(np); s->P[k].vy = real(np);
        s->P[k].vpref = real(np); s->P[k].timer = real(np);
        s->P[k].role = b.take<uint8_t>(np); s->P[k].fsm = b.take<uint8_t>(np);
        s->P[k].state = b.take<uint8_t>(np); s->P[k].active = b.take<uint8_t>(np);
        s->P[k].id = b.take<int32_t>(np); s->P[k].cell = b.take<int32_t>(np);
    }
    for (int k = 0; k < 5; ++k) s->ped_out[k] = real(np);
    for (int k = 0; k < 3; ++k) s->ped_out_u8[k] = b.take<uint8_t>(np);
    for (int k = 0; k < 2; ++k) s->ped_out_i32[k] = b.take<int32_t>(np);
    s->key = b.take<int32_t>(np); s->off = b.take<int32_t>(np); s->cellprev = b.take<int32_t>(2 * np);
    s->perm = b.take<int32_t>(np);
    s->bxy = real(2 * (size_t)np);
    s->count = b.take<int32_t>((size_t)s->nbins + 2); s->start = b.take<int32_t>((size_t)s->nbins + 3);
    s->ghost_zero = b.take<double>(MW); s->ghost_inf = b.take<double>(MW);
    s->chunk_flag = b.take<uint8_t>((size_t)s->march_gx * ((s->grid.ny + 7) / 8));    // room for any R >= 8
    s->nsegx = (s->grid.nx + 63) / 64; s->dry_stride = (size_t)s->nsegx * ((s->grid.ny + 7) / 8 + 2);
    s->dryseg = b.take<uint8_t>(2 * s->dry_stride);
    s->scan_status = b.take<unsigned long long>((size_t)(s->nbins + 1 + SCAN_TILE - 1) / SCAN_TILE + 1);
    return (b.off + 255) & ~size_t(255);
}

int derive_sizes(sim *s, const sim_grid_t *g, int32_t n_peds, const sim_params_t *p)
{
    if (!g || !p) return fail(s, SIM_EINVAL, "null grid or params");
    if (g->nx <= 0 || g->ny <= 0 || (long long)g->nx * g->ny > 0x7fffffffLL)
        return fail(s, SIM_EINVAL, "nx, ny must be positive and nx*ny < 2^31");
    if (!(g->dx > 0) || !(g->dy > 0)) return fail(s, SIM_EINVAL, "dx, dy must be positive");
    if (g->real_bits != 32 && g->real_bits != 64) return fail(s, SIM_EINVAL, "real_bits must be 32 or 64");
    if (n_peds < 0) return fail(s, SIM_EINVAL, "negative pedestrian count");
    if (!(p->R_int > 0)) return fail(s, SIM_EINVAL, "R_int must be positive");
    if (p->n_targets < 1 || p->n_inflow_faces < 0 || p->n_hydro < 0 || p->n_line < 0 || p->n_exit_cells < 0)
        return fail(s, SIM_EINVAL, "bad list length in params");
    s->grid = *g;
    {   // SMs of the current device (148 on a B200; also the value assumed when sizing without a device)
        int dev = 0, n = 0;
        if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0) {
            s->device = dev; s->n_sm = n;
        }
    }
    s->ncell = g->nx * g->ny; s->np = n_peds;
    s->gny = g->slab_ny_global > 0 ? g->slab_ny_global : g->ny;
    s->j0 = g->slab_ny_global > 0 ? g->slab_j0 : 0;
    if (s->j0 < 0 || s->j0 + g->ny > s->gny || (long long)g->nx * s->gny > 0x7fffffffLL)
        return fail(s, SIM_EINVAL, "slab rows [slab_j0, slab_j0 + ny) must lie inside slab_ny_global rows");
    s->pcell = g->nx * s->gny;
    const double dmin = g->dx < g->dy ? g->dx : g->dy;
    s->kbin = (int)std::ceil(p->R_int / dmin); if (s->kbin < 1) s->kbin = 1;     // C26
    s->nbx = (g->nx + s->kbin - 1) / s->kbin; s->nby = (s->gny + s->kbin - 1) / s->kbin;
    s->nbins = s->nbx * s->nby;
    // march kernel geometry: strips of MW columns, chunks of R rows; R shrinks until the grid
    // fills the 148 SMs a few times over
    s->march_gx = (g->nx + MW - 1) / MW;
    // about 10 waves of 148 SMs x 6 resident CTAs (measured on 8192^2 with dry chunks skipped: step 0.582 / 0.574 /
    // 0.568 / 0.566 / 0.569 ms at R = 14 / 19 / 24 / 28 / 32: fewer halo rows and prologues against coarser skipping
    // and a longer tail)
    const long long slots = (long long)s->n_sm * 6;
    s->march_R = (int)(((long long)g->ny * s->march_gx * 2) / (21 * slots));
    if (s->march_R > MARCH_MAX_R) s->march_R = MARCH_MAX_R;
    if (s->march_R < 16) s->march_R = 16;
    if ((long long)s->march_gx * ((g->ny + s->march_R - 1) / s->march_R) < 4 * slots) {
        // few waves: shorter chunks, about two waves of CTAs.  Work per chunk is uneven (dry / wet,
        // solid cells), so dynamic scheduling of more, smaller CTAs beats filling one wave exactly
        // (Config 4, 2048^2: R = 8..12 58.7 us, R = 19 (one wave) 63.3 us, R = 24 74 us)
        s->march_R = (int)(((long long)g->ny * s->march_gx) / (2 * slots));
        if (s->march_R > 16) s->march_R = 16;
        if (s->march_R < 8) s->march_R = 8;
    }
    s->march_gy = (g->ny + s->march_R - 1) / s->march_R;
    s->n_inflow = p->n_inflow_faces; s->n_hydro = p->n_hydro; s->n_line = p->n_line; s->n_targets = p->n_targets;
    return SIM_OK;
}

// launch with the programmatic-serialization attribute (graph mode only; see pdl_wait())
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl, Args... args)
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

template <typename T, int CPT, int STAGES, int MINB>
cudaError_t launch_tmarch(const FloodArgs<T> &fa, dim3 grid, cudaStream_t st, bool pdl)
{
    constexpr size_t dyn = tmarch_dyn_smem<T, STAGES>();      // the opt-in limit is set per device in sim_create (set_smem_attr)
    return launch_pdl(flood_tmarch_kernel<T, CPT, STAGES, MINB>, grid, dim3(MW / CPT), dyn, st, pdl, fa);
}

template <typename T> FloodArgs<T> flood_args(const sim *s)
{
    FloodArgs<T> a{};
    a.nx = s->grid.nx; a.ny = s->grid.ny;
    a.g = (T)s->prm.g; a.inv_dx = (T)(1.0 / s->grid.dx); a.inv_dy = (T)(1.0 / s->grid.dy);
    a.h_dry = (T)s->prm.h_dry; a.cell_area = (T)(s->grid.dx * s->grid.dy);
    a.couple = s->prm.couple_roughness; a.n_cap = s->prm.n_cap;
    for (int k = 0; k < 2; ++k) { a.h[k] = (T *)s->h[k]; a.qx[k] = (T *)s->qx[k]; a.qy[k] = (T *)s->qy[k]; }
    a.zs = (const T *)s->zs; a.n0 = (const T *)s->n0; a.occ = s->occ; a.occ_stride = (size_t)s->ncell;
    for (int k = 0; k < 4; ++k) a.inflow[k] = s->inflow[k];
    a.chunk_flag = s->chunk_flag; a.R = s->march_R;
    a.ghost_zero = (const T *)s->ghost_zero; a.ghost_inf = (const T *)s->ghost_inf; a.ghost_occ = (const uint8_t *)s->ghost_zero;
    a.open_sides = s->prm.open_sides;
    a.dryseg = s->dry_skip ? s->dryseg : nullptr; a.dry_stride = s->dry_stride; a.nsegx = s->nsegx;
    if (s->ngroup > 1) {
        const size_t nx = (size_t)s->grid.nx;
        const sim::Peer *lo = s->grank > 0 ? &s->peer[s->grank - 1] : nullptr, *hi = s->grank + 1 < s->ngroup ? &s->peer[s->grank + 1] : nullptr;
        if (lo) {
            const size_t off = (size_t)(lo->ny - 1) * nx;                  // its last row
            for (int k = 0; k < 2; ++k) { a.halo_h[0][k] = (const T *)lo->h[k] + off; a.halo_qx[0][k] = (const T *)lo->qx[k] + off; a.halo_qy[0][k] = (const T *)lo->qy[k] + off; }
            a.halo_z[0] = (const T *)lo->zs + off;
        }
        if (hi) {                                                          // its first row
            for (int k = 0; k < 2; ++k) { a.halo_h[1][k] = (const T *)hi->h[k]; a.halo_qx[1][k] = (const T *)hi->qx[k]; a.halo_qy[1][k] = (const T *)hi->qy[k]; }
            a.halo_z[1] = (const T *)hi->zs;
        }
    }
    a.ctl = s->ctl;
    return a;
}

template <typename T> PedSoA<T> ped_soa(const sim *s, int k)
{
    PedSoA<T> p{};
    p.x = (T *)s->P[k].x; p.y = (T *)s->P[k].y; p.vx = (T *)s->P[k].vx; p.vy = (T *)s->P[k].vy;
    p.vpref = (T *)s->P[k].vpref; p.timer = (T *)s->P[k].timer;
    p.role = s->P[k].role; p.fsm = s->P[k].fsm; p.state = s->P[k].state; p.active = s->P[k].active;
    p.id = s->P[k].id; p.cell = s->P[k].cell;
    return p;
}

template <typename T> PedArgs<T> ped_args(const sim *s)
{
    PedArgs<T> a{};
    const sim_params_t &p = s->prm;
    a.n = s->np; a.nx = s->grid.nx; a.ny = s->gny;
    a.kbin = s->kbin; a.nbx = s->nbx; a.nby = s->nby; a.nbins = s->nbins;
    a.inv_dx = (T)(1.0 / s->grid.dx); a.inv_dy = (T)(1.0 / s->grid.dy);
    a.h_dry = (T)p.h_dry;
    for (int k = 0; k < 3; ++k) a.hr_edge[k] = (T)p.hr_edges[k];
    for (int k = 0; k < 4; ++k) a.speed_wet[k] = (T)p.speed_wet[k];
    a.inv_tau = (T)(1.0 / p.tau); a.A_s = (T)p.A_s; a.inv_B = (T)(1.0 / p.B_s); a.two_r = (T)(2.0 * p.radius);
    a.R_int = (T)p.R_int; a.R2 = (T)(p.R_int * p.R_int); a.vmax_factor = (T)p.vmax_factor; a.t_pick = (T)p.t_pick; a.t_drop = (T)p.t_drop;
    a.n_targets = p.n_targets; a.exit_target = p.exit_target; a.storage_target = p.storage_target;
    a.drop_target = p.drop_target;
    a.storage_i = p.storage_cell % s->grid.nx; a.storage_j = p.storage_cell / s->grid.nx;
    a.drop_i = p.drop_cell % s->grid.nx; a.drop_j = p.drop_cell / s->grid.nx;
    a.arrive = p.arrive_cells;
    a.A = ped_soa<T>(s, 0); a.B = ped_soa<T>(s, 1);
    a.key = s->key; a.off = s->off; a.perm = s->perm; a.count = s->count; a.start = s->start; a.cellprev = s->cellprev;
    a.mask = s->mask; a.nav = s->nav;
    a.cellprev_stride = (size_t)s->np; a.pipelined = 0;
    a.bxy = (VecN<T, 2> *)s->bxy;
    a.c_exp1 = (T)(2.0 * p.radius / p.B_s * 1.4426950408889634 + std::log2(p.A_s));   // A e^{(2r-d)/B} = 2^{c1 + c2 d}
    a.c_exp2 = (T)(-1.4426950408889634 / p.B_s);
    // where the flood state of a cell lives: one slab (this handle's own grid) unless linked (8f-4)
    const int ng = s->ngroup > 0 ? s->ngroup : 1;
    sim::Peer self; self.j0 = s->j0; self.ny = s->grid.ny; self.zs = s->zs; self.occ = s->occ; self.ctl = s->ctl;
    for (int k = 0; k < 2; ++k) { self.h[k] = s->h[k]; self.qx[k] = s->qx[k]; self.qy[k] = s->qy[k]; }
    a.slab.n = ng; a.slab.rows = ng > 1 ? s->peer[0].ny : s->gny;
    for (int r = 0; r < ng; ++r) {
        const sim::Peer *q = ng > 1 ? &s->peer[r] : &self;
        const ptrdiff_t off = (ptrdiff_t)q->j0 * s->grid.nx;
        for (int k = 0; k < 2; ++k) {
            a.slab.h[k][r] = (const T *)q->h[k] - off; a.slab.qx[k][r] = (const T *)q->qx[k] - off; a.slab.qy[k][r] = (const T *)q->qy[k] - off;
            a.slab.occ[k][r] = q->occ + (size_t)k * ((size_t)q->ny * s->grid.nx) - off;
        }
    }
    a.ctl = s->ctl;
    return a;
}

template <typename T> TailArgs<T> tail_args(const sim *s)
{
    TailArgs<T> a{};
    a.ctl = s->ctl; a.line_cells = s->line_cells;
    {
        const int ng = s->ngroup > 0 ? s->ngroup : 1;
        a.slab_rows = ng > 1 ? s->peer[0].ny : s->gny; a.nx = s->grid.nx; a.n_slabs = ng;
        for (int r = 0; r < ng; ++r) {
            void *zs = ng > 1 ? s->peer[r].zs : s->zs; const int j0 = ng > 1 ? s->peer[r].j0 : s->j0;
            a.zs_tab[r] = (T *)zs - (ptrdiff_t)j0 * s->grid.nx;
        }
    }
    a.n_line = s->n_line; a.bags_per_cell_layer = s->prm.bags_per_cell_layer; a.n_layers = s->prm.n_layers;
    a.layer_thickness = (T)s->prm.layer_thickness;
    a.hydro_t = s->hydro_t; a.hydro_q = s->hydro_q; a.n_hydro = s->n_hydro;
    a.inv_inflow_length = s->inflow_length > 0 ? 1.0 / s->inflow_length : 0.0;
    a.A = ped_soa<T>(s, 0); a.np = s->np; a.n_doors = s->prm.n_doors;
    for (int d = 0; d < s->prm.n_doors; ++d) a.door_cells[d] = s->door_cells[d];
    a.door_credit = s->door_credit;
    a.spawn_rate = s->prm.spawn_rate; a.vpref_lo = s->prm.spawn_vpref_lo; a.vpref_hi = s->prm.spawn_vpref_hi;
    a.dx = s->grid.dx; a.dy = s->grid.dy; a.target_population = s->prm.target_population;
    a.seed_lo = (unsigned)(s->prm.spawn_seed & 0xffffffffull); a.seed_hi = (unsigned)(s->prm.spawn_seed >> 32);
    return a;
}

// ---- launch helpers.  Kernel arguments are the same every step: the ping-pong parity, dt, t,
// halt live in the device control block.
template <typename T> PedArgs<T> ped_args_full(const sim *s, int pipelined)
{
    PedArgs<T> pa = ped_args<T>(s);
    for (int e = 0; e < s->prm.n_exit_cells; ++e) { pa.exit_i[e] = s->exit_i[e]; pa.exit_j[e] = s->exit_j[e]; }
    pa.n_exit = s->prm.n_exit_cells;
    pa.n_doors = s->prm.n_doors;
    for (int d = 0; d < s->prm.n_doors; ++d) {
        pa.door_i[d] = s->door_cells[d] % s->grid.nx; pa.door_j[d] = s->door_cells[d] / s->grid.nx;
        pa.door_target[d] = s->door_target[d];
    }
    pa.pipelined = pipelined;
    pa.pdl_early = s->np >= 65536;
    pa.occ_in_scatter = s->np < 65536;   // small crowds are launch-bound: four dependent launches per step instead of five   // measured: pre-scheduling the chain pays on Config 5 (-1.5 %), costs on Configs 1-3 (+8 %)
    return pa;
}

struct Marks {                                        // profiling mode only: an event before each launch
    cudaEvent_t *ev; int k; cudaStream_t st;
    void operator()() { if (ev) cudaEventRecord(ev[k++], st); }
};

// (B)+(O) of the step that comes NEXT: count -> scan -> scatter -> N_p per cell.  It needs the
// pedestrians of that step only, so in graph mode it runs beside the flood kernel of the step
// before (pipelined = 1: it fills the N_p buffer the flood kernel is not reading).
template <typename T> int enqueue_bin_chain(sim *s, cudaStream_t st, int pipelined, Marks &mark, bool counted = false)
{
    PedArgs<T> pa = ped_args_full<T>(s, pipelined);
    const int nb = (s->np + 255) / 256, n_items = s->nbins + 1;
    const bool pdl = s->pdl && !mark.ev;              // graph mode: each kernel may start under the tail of the one before
    mark();
    if (!counted) CU(launch_pdl(ped_bin_count_kernel<T>, dim3(nb), dim3(256), 0, st, pdl && pipelined, pa, 1));
    mark();
    CU(launch_pdl(scan_bins_kernel, dim3((n_items + SCAN_TILE - 1) / SCAN_TILE), dim3(SCAN_THREADS), 0, st, pdl,
                  s->count, s->start, n_items, s->scan_status, s->ctl, pipelined, pa.pdl_early));
    if (s->deterministic) {                           // bins ordered by original id (see ped_rank_kernel)
        CU(launch_pdl(ped_perm_kernel<T>, dim3(nb), dim3(256), 0, st, pdl, pa));
        CU(launch_pdl(ped_rank_kernel<T>, dim3(nb), dim3(256), 0, st, pdl, pa));
    }
    mark();
    CU(launch_pdl(ped_scatter_kernel<T>, dim3(nb), dim3(256), 0, st, pdl, pa));
    mark();
    if (!pa.occ_in_scatter) CU(launch_pdl(ped_occ_kernel<T>, dim3(nb), dim3(256), 0, st, pdl, pa));
    CU(cudaGetLastError());
    return SIM_OK;
}

template <typename T> int launch_flood(sim *s, cudaStream_t st, bool pdl)
{
    FloodArgs<T> fa = flood_args<T>(s);
    if (s->flood_variant == 5) {                     // second order (flood_order = 2)
        dim3 grid((s->grid.nx + MTX - 1) / MTX, (s->grid.ny + MTY - 1) / MTY);
        CU(launch_pdl(flood_muscl_kernel<T>, grid, dim3(MTX, MTY), sizeof(MusclSmem<T>), st, pdl, fa));
    } else if (s->flood_variant == 4) {
        CU((launch_tmarch<T, 2, 4, 6>(fa, dim3(s->march_gx, s->march_gy), st, pdl)));
    } else if (s->flood_variant == 3) {
        CU(launch_pdl(flood_march2_kernel<T, 2>, dim3(s->march_gx, s->march_gy), dim3(MW / 2), 0, st, pdl, fa));
    } else if (s->flood_variant == 2) {
        CU(launch_pdl(flood_march_kernel<T>, dim3(s->march_gx, s->march_gy), dim3(MW), 0, st, pdl, fa));
    } else if (s->flood_variant == 1) {
        dim3 grid((s->grid.nx + TX - 1) / TX, (s->grid.ny + TY - 1) / TY);
        CU(launch_pdl(flood_tile_kernel<T>, grid, dim3(FLOOD_TILE_THREADS), sizeof(TileSmem<T>), st, pdl, fa));
    } else {
        dim3 blk(32, 8), grid((s->grid.nx + 31) / 32, (s->grid.ny + 7) / 8);
        CU(launch_pdl(flood_cell_kernel<T>, grid, blk, 0, st, pdl, fa));
    }
    return SIM_OK;
}

// ONE coupled step n on `st`, given that the binning chain of step n has run (sim::binned):
//     pedestrian step n | flood step n  ->  tail n ;   binning chain of step n+1
// Every read of step n is at level n, so the pedestrian step and the flood step are independent;
// the binning chain of step n+1 needs the pedestrian step n only.  In graph mode (fork) the
// pedestrian kernels form a second branch: ped_step(n) -> chain(n+1) beside flood(n); tail(n)
// joins flood(n) and ped_step(n) (deposits), flood(n+1) joins tail(n) and chain(n+1).
template <typename T> int enqueue_step(sim *s, cudaStream_t st, bool first, cudaEvent_t *ev = nullptr)
{
    Marks mark{ev, 0, st};
    const bool peds = s->np > 0;
    const bool fork = !ev && peds && s->overlap;
    cudaStream_t sp = fork ? s->stream2 : st;
    if (peds) {
        if (fork) {
            if (first) { CU(cudaEventRecord(s->ev_fork, st)); CU(cudaStreamWaitEvent(sp, s->ev_fork, 0)); }
            else CU(cudaStreamWaitEvent(sp, s->ev_tail, 0));
        }
        mark();
        CU(launch_pdl(ped_step_kernel<T>, dim3((s->np + PED_THREADS - 1) / PED_THREADS), dim3(PED_THREADS), 0, sp, s->pdl && !ev, ped_args_full<T>(s, 0), fork ? 1 : 0));
        if (fork) {
            CU(cudaEventRecord(s->ev_ped, sp));
            if (!first) CU(cudaStreamWaitEvent(st, s->ev_occ, 0));     // N_p of this step, filled beside the step before
        }
    } else mark.k = 1;
    mark();
    {
        int rc = launch_flood<T>(s, st, s->pdl && !ev);
        if (rc != SIM_OK) return rc;
    }
    if (fork) {
        int rc = enqueue_bin_chain<T>(s, sp, 1, mark, true);             // counted inside ped_step
        if (rc != SIM_OK) return rc;
        CU(cudaEventRecord(s->ev_occ, sp));
        CU(cudaStreamWaitEvent(st, s->ev_ped, 0));
    }
    mark();
    CU(launch_pdl(tail_kernel<T>, dim3(1), dim3(32), 0, st, s->pdl && !ev, tail_args<T>(s), 0));
    if (fork) CU(cudaEventRecord(s->ev_tail, st));
    if (peds && !fork) {
        int rc = enqueue_bin_chain<T>(s, st, 0, mark);               // after the tail: ctl->parity is that of step n+1
        if (rc != SIM_OK) return rc;
    }
    mark();
    CU(cudaGetLastError());
    return SIM_OK;
}

// the binning chain of the upcoming step, when nothing has prepared it (first step, state re-injected)
template <typename T> int prepare_bins(sim *s)
{
    if (s->np > 0 && !s->binned) {
        Marks none{nullptr, 0, s->stream};
        int rc = enqueue_bin_chain<T>(s, s->stream, 0, none);
        if (rc != SIM_OK) return rc;
    }
    s->binned = true;
    return SIM_OK;
}

// n steps launched kernel by kernel with an event before each launch: per-kernel device time
template <typename T> int step_profiled(sim *s, int64_t n, double *ms)
{
    constexpr int NE = 8, BATCH = 64;
    static const int slot_of[NE - 1] = {3, 4, 5, 0, 1, 2, 6};       // launch order -> kernel_ms index
    std::vector<cudaEvent_t> ev(NE * BATCH, nullptr);
    struct Cleanup { std::vector<cudaEvent_t> &v; ~Cleanup() { for (auto e : v) if (e) cudaEventDestroy(e); } } cleanup{ev};
    for (auto &e : ev) CU(cudaEventCreate(&e));
    for (int k = 0; k < 8; ++k) ms[k] = 0.0;
    int rc = prepare_bins<T>(s);
    while (n > 0 && rc == SIM_OK) {
        const int m = (int)(n < BATCH ? n : BATCH);
        for (int i = 0; i < m && rc == SIM_OK; ++i) rc = enqueue_step<T>(s, s->stream, false, &ev[(size_t)i * NE]);
        if (rc != SIM_OK) break;
        cudaError_t e = cudaStreamSynchronize(s->stream);
        if (e != cudaSuccess) { rc = fail(s, SIM_ECUDA, cudaGetErrorString(e)); break; }
        const int first = s->np > 0 ? 0 : 1, last = s->np > 0 ? NE - 1 : 3;
        for (int i = 0; i < m; ++i)
            for (int k = first; k < last; ++k) {
                float t = 0.f;
                cudaEventElapsedTime(&t, ev[(size_t)i * NE + k], ev[(size_t)i * NE + k + 1]);
                ms[slot_of[k]] += t;
            }
        n -= m;
    }
    return rc;
}

void drop_graphs(sim *s)
{
    for (auto &g : s->graph) { if (g) cudaGraphExecDestroy(g); g = nullptr; }
}

template <typename T> int build_graph(sim *s, int level)
{
    const int reps = 1 << level;
    cudaGraph_t g = nullptr;
    CU(cudaStreamBeginCapture(s->cap_stream, cudaStreamCaptureModeThreadLocal));
    int rc = SIM_OK;
    for (int r = 0; r < reps && rc == SIM_OK; ++r) rc = enqueue_step<T>(s, s->cap_stream, r == 0);
    if (rc == SIM_OK && s->np > 0 && s->overlap && cudaStreamWaitEvent(s->cap_stream, s->ev_occ, 0) != cudaSuccess)
        rc = fail(s, SIM_ECUDA, "graph capture: join");
    cudaError_t e = cudaStreamEndCapture(s->cap_stream, &g);
    if (rc != SIM_OK) { if (g) cudaGraphDestroy(g); return rc; }
    if (e != cudaSuccess) return fail(s, SIM_ECUDA, std::string("graph capture: ") + cudaGetErrorString(e));
    cudaGraphExec_t ex = nullptr;
    e = cudaGraphInstantiate(&ex, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) return fail(s, SIM_ECUDA, std::string("graph instantiate: ") + cudaGetErrorString(e));
    e = cudaGraphUpload(ex, s->stream);              // so that the first replay of a ladder level costs what every replay costs
    if (e != cudaSuccess) { cudaGraphExecDestroy(ex); return fail(s, SIM_ECUDA, std::string("graph upload: ") + cudaGetErrorString(e)); }
    s->graph[level] = ex;
    return SIM_OK;
}

template <typename T> int refresh_dt(sim *s)      // lambda of the state in place -> dt, q_in, halt
{
    flood_chunk_flags_kernel<T><<<dim3(s->march_gx, s->march_gy), 256, 0, s->stream>>>((const T *)s->zs, s->grid.nx, s->grid.ny, s->march_R, s->chunk_flag);
    flood_lambda_kernel<T><<<592, 256, 0, s->stream>>>(flood_args<T>(s));
    tail_kernel<T><<<1, 32, 0, s->stream>>>(tail_args<T>(s), 1);
    CU(cudaGetLastError());
    return SIM_OK;
}

// opt-in dynamic shared memory of the kernels that need it, on the handle's device (the attribute is per device)
template <typename T> int set_smem_attr(sim *s)
{
    CU(cudaFuncSetAttribute(flood_tile_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(TileSmem<T>)));
    CU(cudaFuncSetAttribute(flood_tmarch_kernel<T, 2, 4, 6>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tmarch_dyn_smem<T, 4>()));
    CU(cudaFuncSetAttribute(flood_muscl_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(MusclSmem<T>)));
    return SIM_OK;
}

#define DISPATCH(s, fn, ...) ((s)->grid.real_bits == 64 ? fn<double>(__VA_ARGS__) : fn<float>(__VA_ARGS__))

int copy_out(sim *s, void *dst, const void *src, size_t bytes)
{
    if (!dst || !bytes) return SIM_OK;
    CU(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDefault, s->stream));
    return SIM_OK;
}

int upload(sim *s, void *dst, const void *src, size_t bytes)
{
    if (!bytes) return SIM_OK;
    if (src) CU(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, s->stream));
    else CU(cudaMemsetAsync(dst, 0, bytes, s->stream));
    return SIM_OK;
}

// host-side preparation of one real array with solids applied
template <typename T> T solid_value() { return std::numeric_limits<T>::infinity(); }

template <typename T>
void make_zs(const T *z, const uint8_t *mask, size_t n, std::vector<T> &out)
{
    out.resize(n);
    for (size_t c = 0; c < n; ++c) out[c] = (mask && mask[c]) ? (T)INFINITY : z[c];
}

template <typename T>
void make_q(const T *h0, const T *u0, const uint8_t *mask, size_t n, std::vector<T> &out)
{
    out.assign(n, (T)0);
    if (h0 && u0)
        for (size_t c = 0; c < n; ++c) out[c] = (mask && mask[c]) ? (T)0 : h0[c] * u0[c];   // conserved (C8)
}

template <typename T>
double default_dt_max(const sim_peds_t *peds, const sim_params_t *p, double dmin)
{
    double vm = 1.8;                                        // C10
    const T *vp = peds ? (const T *)peds->v_pref : nullptr;
    for (int i = 0; vp && i < peds->n; ++i) if ((double)vp[i] > vm) vm = (double)vp[i];
    for (int k = 0; k < 4; ++k) if (p->speed_wet[k] > vm) vm = p->speed_wet[k];
    return std::fmin(1.0, dmin / (p->vmax_factor * vm));
}

template <typename T>
int upload_state(sim *s, const sim_topo_t *topo, const void *manning, const sim_peds_t *peds, const sim_params_t *p)
{
    const size_t nc = (size_t)s->ncell, rs = sizeof(T);
    // a row slab (8f-4) is given the arrays of the WHOLE grid and takes its rows of the flood fields
    const size_t so = (size_t)s->j0 * s->grid.nx;
    sim_topo_t cut = *topo;
    cut.z = (const T *)topo->z + so; cut.mask = topo->mask ? topo->mask + so : nullptr;
    cut.h0 = topo->h0 ? (const T *)topo->h0 + so : nullptr; cut.u0 = topo->u0 ? (const T *)topo->u0 + so : nullptr;
    cut.v0 = topo->v0 ? (const T *)topo->v0 + so : nullptr;
    const uint8_t *mask_all = topo->mask;
    topo = &cut; manning = (const T *)manning + so;
    std::vector<T> tmp;
    make_zs<T>((const T *)topo->z, topo->mask, nc, tmp);
    if (upload(s, s->zs, tmp.data(), nc * rs)) return SIM_ECUDA;
    CU(cudaStreamSynchronize(s->stream));
    {   // the row beyond the domain edge: solid cells (ghost_zero stays at the workspace's zeros)
        std::vector<T> inf(MW, solid_value<T>());
        if (upload(s, s->ghost_inf, inf.data(), MW * rs)) return SIM_ECUDA;
        CU(cudaStreamSynchronize(s->stream));
    }
    if (upload(s, s->z0, topo->z, nc * rs)) return SIM_ECUDA;
    if (upload(s, s->n0, manning, nc * rs)) return SIM_ECUDA;
    if (s->np > 0 && upload(s, s->mask, mask_all, (size_t)s->pcell)) return SIM_ECUDA;      // the pedestrians' mask: whole grid
    // depth: zero inside solids
    if (topo->h0) {
        tmp.resize(nc);
        const T *h0 = (const T *)topo->h0;
        for (size_t c = 0; c < nc; ++c) tmp[c] = (topo->mask && topo->mask[c]) ? (T)0 : h0[c];
        if (upload(s, s->h[0], tmp.data(), nc * rs)) return SIM_ECUDA;
        CU(cudaStreamSynchronize(s->stream));
    } else if (upload(s, s->h[0], nullptr, nc * rs)) return SIM_ECUDA;
    make_q<T>((const T *)topo->h0, (const T *)topo->u0, topo->mask, nc, tmp);
    if (upload(s, s->qx[0], tmp.data(), nc * rs)) return SIM_ECUDA;
    CU(cudaStreamSynchronize(s->stream));
    make_q<T>((const T *)topo->h0, (const T *)topo->v0, topo->mask, nc, tmp);
    if (upload(s, s->qy[0], tmp.data(), nc * rs)) return SIM_ECUDA;
    CU(cudaStreamSynchronize(s->stream));
    // pedestrians: buffer A in original order
    const size_t np = (size_t)s->np;
    if (np) {
        if (upload(s, s->P[0].x, peds->x, np * rs) || upload(s, s->P[0].y, peds->y, np * rs) ||
            upload(s, s->P[0].vx, peds->vx, np * rs) || upload(s, s->P[0].vy, peds->vy, np * rs) ||
            upload(s, s->P[0].vpref, peds->v_pref, np * rs) || upload(s, s->P[0].role, peds->role, np))
            return SIM_ECUDA;
        std::vector<uint8_t> fsm(np), act(np, 1);
        if (peds->active) for (size_t i = 0; i < np; ++i) act[i] = peds->active[i] ? 1 : 0;
        std::vector<int32_t> id(np), neg(np, -1);
        for (size_t i = 0; i < np; ++i) {
            fsm[i] = (peds->role && peds->role[i]) ? SIM_FSM_TO_STORAGE : SIM_FSM_EVACUATE;
            id[i] = (int32_t)i;
        }
        if (upload(s, s->P[0].fsm, fsm.data(), np) || upload(s, s->P[0].active, act.data(), np) ||
            upload(s, s->P[0].id, id.data(), np * 4) || upload(s, s->cellprev, neg.data(), np * 4) ||
            upload(s, s->cellprev + np, neg.data(), np * 4))
            return SIM_ECUDA;
        CU(cudaStreamSynchronize(s->stream));
    }
    (void)p;
    return SIM_OK;
}

}  // namespace

// ================================================================================ C ABI

extern "C" int sim_workspace_bytes(const sim_grid_t *grid, int32_t n_peds, const sim_params_t *params, size_t *bytes)
{
    sim tmp;
    if (!bytes) return fail(nullptr, SIM_EINVAL, "bytes is NULL");
    int rc = derive_sizes(&tmp, grid, n_peds, params);
    if (rc != SIM_OK) { g_create_error = tmp.err; return rc; }
    Bump b; b.dry = true;
    *bytes = layout(&tmp, b);
    return SIM_OK;
}

extern "C" int sim_create(const sim_grid_t *grid, const sim_topo_t *topo, const void *manning,
                          const sim_peds_t *peds, const sim_params_t *p, void *workspace,
                          void *cuda_stream, sim_t **out)
{
    if (!out) return fail(nullptr, SIM_EINVAL, "out is NULL");
    *out = nullptr;
    sim *s = new sim;
    auto bail = [&](int rc) { g_create_error = s->err; sim_destroy(s); return rc; };
    const int32_t n_peds = peds ? peds->n : 0;
    int rc = derive_sizes(s, grid, n_peds, p);
    if (rc != SIM_OK) return bail(rc);
    if (!topo || !topo->z || !manning) return bail(fail(s, SIM_EINVAL, "z and manning are required"));
    if (n_peds > 0 && (!peds->x || !peds->y || !peds->vx || !peds->vy || !peds->v_pref))
        return bail(fail(s, SIM_EINVAL, "pedestrian arrays are required when n > 0"));
    if (n_peds > 0 && !p->nav_dir) return bail(fail(s, SIM_EINVAL, "nav_dir is required"));
    if (p->n_cap < 0 || p->n_cap > 255) return bail(fail(s, SIM_EINVAL, "n_cap must be in [0, 255]"));
    if (p->n_exit_cells > 16) return bail(fail(s, SIM_EINVAL, "at most 16 exit cells"));
    if (!(p->tau > 0) || !(p->B_s > 0) || !(p->g > 0) || !(p->cfl > 0))
        return bail(fail(s, SIM_EINVAL, "tau, B_s, g, cfl must be positive"));
    if (!(p->h_dry > 0) || (grid->real_bits == 32 && p->h_dry < 1.2e-38))
        return bail(fail(s, SIM_EINVAL, "h_dry must be positive (and a normal number in the storage precision): depths are divided by max(h, h_dry)"));
    if (p->open_sides < 0 || p->open_sides > 15) return bail(fail(s, SIM_EINVAL, "open_sides is a mask of the four sides"));
    if (p->n_doors < 0 || p->n_doors > 16) return bail(fail(s, SIM_EINVAL, "at most 16 doors"));
    if (p->n_doors > 0) {
        if (!p->door_cells || !p->door_target) return bail(fail(s, SIM_EINVAL, "door_cells and door_target are required when n_doors > 0"));
        if (!(p->spawn_rate >= 0) || p->target_population < 0 || !(p->spawn_vpref_hi >= p->spawn_vpref_lo) || !(p->spawn_vpref_lo > 0))
            return bail(fail(s, SIM_EINVAL, "spawn_rate, target_population >= 0 and 0 < spawn_vpref_lo <= spawn_vpref_hi are required"));
        for (int d = 0; d < p->n_doors; ++d) {
            const int c = p->door_cells[d];
            if (c < 0 || c >= s->pcell || (topo->mask && topo->mask[c])) return bail(fail(s, SIM_EINVAL, "door cell out of range or solid"));
            if (p->door_target[d] < 0 || p->door_target[d] >= p->n_targets) return bail(fail(s, SIM_EINVAL, "door target out of range"));
        }
    }
    if (p->flood_order < 0 || p->flood_order > 2) return bail(fail(s, SIM_EINVAL, "flood_order must be 0, 1 (first order, the paper's scheme) or 2 (MUSCL-Hancock)"));
    if (!(p->A_s > 0) || !(p->radius >= 0) || !(p->vmax_factor > 0))
        return bail(fail(s, SIM_EINVAL, "A_s and vmax_factor must be positive, radius non-negative"));
    if (workspace && ((uintptr_t)workspace % 256) != 0)
        return bail(fail(s, SIM_EINVAL, "workspace must be 256-byte aligned (TMA row copies need 16-byte aligned rows)"));
    if (p->exit_target < 0 || p->exit_target >= p->n_targets || p->storage_target < 0 ||
        p->storage_target >= p->n_targets || p->drop_target < 0 || p->drop_target >= p->n_targets)
        return bail(fail(s, SIM_EINVAL, "target index out of range"));
    const int nx = grid->nx, ny = grid->ny, gny = s->gny, j0 = s->j0;      // cell indices are those of the whole grid
    auto cell_ok = [&](int c) { return c >= 0 && c < nx * gny; };
    for (int e = 0; e < p->n_exit_cells; ++e)
        if (!cell_ok(p->exit_cells[e])) return bail(fail(s, SIM_EINVAL, "exit cell out of range"));
    if (!cell_ok(p->storage_cell) || !cell_ok(p->drop_cell)) return bail(fail(s, SIM_EINVAL, "storage/drop cell out of range"));
    for (int k = 0; k < p->n_line; ++k) {
        if (!cell_ok(p->line_cells[k])) return bail(fail(s, SIM_EINVAL, "barrier cell out of range"));
        if (topo->mask && topo->mask[p->line_cells[k]]) return bail(fail(s, SIM_EINVAL, "barrier cell is solid"));
        s->line_row_max = std::max(s->line_row_max, p->line_cells[k] / nx);
    }
    if (p->n_line > 0 && p->n_layers > 0 && p->bags_per_cell_layer < 1)
        return bail(fail(s, SIM_EINVAL, "bags_per_cell_layer must be >= 1"));
    std::vector<uint8_t> infl[4];
    infl[0].assign(ny, 0); infl[1].assign(ny, 0); infl[2].assign(nx, 0); infl[3].assign(nx, 0);
    s->inflow_length = 0.0;
    for (int f = 0; f < p->n_inflow_faces; ++f) {
        const int c = p->inflow_cell[f], side = p->inflow_side[f];
        if (!cell_ok(c) || side > 3) return bail(fail(s, SIM_EINVAL, "inflow face out of range"));
        const int i = c % nx, j = c / nx;
        const bool on_edge = (side == SIM_SIDE_W && i == 0) || (side == SIM_SIDE_E && i == nx - 1) ||
                             (side == SIM_SIDE_S && j == 0) || (side == SIM_SIDE_N && j == gny - 1);
        if (!on_edge) return bail(fail(s, SIM_EINVAL, "inflow faces must lie on the domain edge (C14)"));
        if (topo->mask && topo->mask[c]) return bail(fail(s, SIM_EINVAL, "inflow face on a solid cell: its share of Q(t) would be lost"));
        s->inflow_length += side < 2 ? grid->dy : grid->dx;                 // of the whole grid: q_in = Q / length
        if (j < j0 || j >= j0 + ny) continue;                                // another slab's face
        uint8_t &m = infl[side][side < 2 ? j - j0 : i];
        if (m == 255) return bail(fail(s, SIM_EINVAL, "too many inflow faces on one cell side"));
        m += 1;
    }
    for (int k = 1; k < p->n_hydro; ++k)
        if (!(p->hydro_t[k] > p->hydro_t[k - 1])) return bail(fail(s, SIM_EINVAL, "hydro_t must increase"));

    s->prm = *p;
    for (int e = 0; e < p->n_exit_cells; ++e) { s->exit_i[e] = p->exit_cells[e] % nx; s->exit_j[e] = p->exit_cells[e] / nx; }
    if (!(s->prm.dt_max > 0)) {
        const double dmin = grid->dx < grid->dy ? grid->dx : grid->dy;
        s->prm.dt_max = grid->real_bits == 64 ? default_dt_max<double>(peds, p, dmin) : default_dt_max<float>(peds, p, dmin);
    }
    s->flood_variant = ((long long)nx * ny >= (1ll << 22)) ? (nx % 16 == 0 ? 4 : nx % 2 == 0 ? 3 : 2) : (nx % 4 == 0) ? 1 : 0;
    if (p->open_sides) s->flood_variant = 0;       // open edges: the one-thread-per-cell kernel (and the MUSCL kernel)
    if (p->flood_order == 2) s->flood_variant = 5;
    for (int d = 0; d < p->n_doors; ++d) { s->door_cells[d] = p->door_cells[d]; s->door_target[d] = p->door_target[d]; }
    // doors: newcomers are placed by the tail kernel, so the binning of the next step must come after it
    if (p->n_doors > 0) s->overlap = 0;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
        return bail(fail(s, SIM_ECUDA, "no CUDA device: this library has no CPU fallback"));
    s->stream = (cudaStream_t)cuda_stream;
    Bump b; b.dry = true;
    s->ws_bytes = layout(s, b);
    if (workspace) { s->ws = workspace; s->own_ws = false; }
    else {
        if (cudaMalloc(&s->ws, s->ws_bytes) != cudaSuccess) { s->ws = nullptr; return bail(fail(s, SIM_ENOMEM, "cudaMalloc of the workspace failed")); }
        s->own_ws = true;
    }
    b = Bump(); b.dry = false; b.base = (char *)s->ws;
    layout(s, b);
    auto run = [&]() -> int {
        CU(cudaMemsetAsync(s->ws, 0, s->ws_bytes, s->stream));
        CU(cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&s->stream2, cudaStreamNonBlocking));
        CU(cudaEventCreateWithFlags(&s->ev_fork, cudaEventDisableTiming));
        CU(cudaEventCreateWithFlags(&s->ev_ped, cudaEventDisableTiming));
        CU(cudaEventCreateWithFlags(&s->ev_occ, cudaEventDisableTiming));
        CU(cudaEventCreateWithFlags(&s->ev_tail, cudaEventDisableTiming));
        int r = DISPATCH(s, upload_state, s, topo, manning, peds, p);
        if (r != SIM_OK) return r;
        for (int k = 0; k < 4; ++k) if (upload(s, s->inflow[k], infl[k].data(), infl[k].size())) return SIM_ECUDA;
        if (s->np > 0 && upload(s, s->nav, p->nav_dir, (size_t)p->n_targets * s->pcell)) return SIM_ECUDA;
        if (p->n_line && upload(s, s->line_cells, p->line_cells, (size_t)p->n_line * 4)) return SIM_ECUDA;
        if (p->n_hydro && (upload(s, s->hydro_t, p->hydro_t, (size_t)p->n_hydro * 8) ||
                           upload(s, s->hydro_q, p->hydro_q, (size_t)p->n_hydro * 8))) return SIM_ECUDA;
        Ctl c{};
        c.t = 0.0; c.dt = 0.0; c.t_end = s->prm.t_end; c.dt_max = s->prm.dt_max; c.cfl = s->prm.cfl;
        c.complete = (p->n_line <= 0 || p->n_layers <= 0) ? 1 : 0;
        c.scan_epoch = 1;
        c.pair_c1 = (float)(2.0 * p->radius / p->B_s * 1.4426950408889634 + std::log2(p->A_s));
        c.pair_c2 = (float)(-1.4426950408889634 / p->B_s);
        CU(cudaMemcpyAsync(s->ctl, &c, sizeof c, cudaMemcpyHostToDevice, s->stream));
        CU(cudaStreamSynchronize(s->stream));
        r = DISPATCH(s, set_smem_attr, s);
        if (r != SIM_OK) return r;
        r = DISPATCH(s, refresh_dt, s);
        if (r != SIM_OK) return r;
        CU(cudaStreamSynchronize(s->stream));
        return SIM_OK;
    };
    rc = run();
    if (rc != SIM_OK) return bail(rc);
    *out = s;
    return SIM_OK;
}

extern "C" int sim_step(sim_t *s, int64_t n)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    if (n < 0) return fail(s, SIM_EINVAL, "negative step count");
    if (s->ngroup > 1) return fail(s, SIM_EINVAL, "a linked row slab steps with sim_slab_step");
    if (n == 0) return SIM_OK;
    {
        int rc = DISPATCH(s, prepare_bins, s);
        if (rc != SIM_OK) return rc;
    }
    // all graphs are captured at the first call (a few ms, once), never inside a later, timed call
    for (int level = 0; level < GRAPH_LEVELS; ++level)
        if (!s->graph[level]) {
            int rc = DISPATCH(s, build_graph, s, level);
            if (rc != SIM_OK) return rc;
        }
    // n = sum of powers of two: the largest graph repeatedly, then one replay per set bit
    for (int level = GRAPH_LEVELS - 1; level >= 0 && n > 0; --level) {
        const int64_t reps = (int64_t)1 << level;
        if (n < reps) continue;
        while (n >= reps) {
            CU(cudaGraphLaunch(s->graph[level], s->stream));
            n -= reps;
            if (level < GRAPH_LEVELS - 1) break;
        }
    }
    return SIM_OK;
}

extern "C" int sim_step_profiled(sim_t *s, int64_t n, double *kernel_ms)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    if (n < 0 || !kernel_ms) return fail(s, SIM_EINVAL, "bad arguments");
    return DISPATCH(s, step_profiled, s, n, kernel_ms);
}

extern "C" int sim_kernels_per_step(const sim_t *s) { return s ? (s->np > 0 ? (s->overlap ? 6 : 7) - (s->np < 65536 ? 1 : 0) + (s->deterministic ? 2 : 0) : 2) : 0; }

extern "C" int sim_set_march_rows(sim_t *s, int32_t rows)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    if (rows < 8 || rows > MARCH_MAX_R) return fail(s, SIM_EINVAL, "rows per chunk must be in [8, 64]");
    CU(cudaStreamSynchronize(s->stream));
    s->march_R = rows;
    s->march_gy = (s->grid.ny + rows - 1) / rows;
    drop_graphs(s);
    CU(cudaMemsetAsync(s->dryseg, 0, 2 * s->dry_stride, s->stream));       // the flags are per chunk row of R rows
    if (s->grid.real_bits == 32)
        flood_chunk_flags_kernel<float><<<dim3(s->march_gx, s->march_gy), 256, 0, s->stream>>>((const float *)s->zs, s->grid.nx, s->grid.ny, s->march_R, s->chunk_flag);
    else
        flood_chunk_flags_kernel<double><<<dim3(s->march_gx, s->march_gy), 256, 0, s->stream>>>((const double *)s->zs, s->grid.nx, s->grid.ny, s->march_R, s->chunk_flag);
    CU(cudaGetLastError());
    return SIM_OK;
}

extern "C" int sim_set_overlap(sim_t *s, int32_t on)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    CU(cudaStreamSynchronize(s->stream));
    if (on && s->prm.n_doors > 0) return fail(s, SIM_EINVAL, "with doors the step is one chain: newcomers are placed before the binning of the next step");
    s->overlap = on ? 1 : 0;
    drop_graphs(s);
    return SIM_OK;
}

// ---- row slabs
namespace {

template <typename T> int slab_refresh(sim *const *h, int n)
{
    SlabCtls t{}; t.n = n;
    for (int r = 0; r < n; ++r) {
        sim *s = h[r];
        DeviceGuard g(s);
        t.c[r] = s->ctl;
        flood_chunk_flags_kernel<T><<<dim3(s->march_gx, s->march_gy), 256, 0, s->stream>>>((const T *)s->zs, s->grid.nx, s->grid.ny, s->march_R, s->chunk_flag);
        flood_lambda_kernel<T><<<592, 256, 0, s->stream>>>(flood_args<T>(s));
        CU(cudaGetLastError());
        CU(cudaStreamSynchronize(s->stream));
    }
    {
        sim *s = h[0];
        DeviceGuard g(s);
        slab_lambda_kernel<<<1, 32, 0, s->stream>>>(t);
        CU(cudaGetLastError());
        CU(cudaStreamSynchronize(s->stream));
    }
    for (int r = 0; r < n; ++r) {
        sim *s = h[r];
        DeviceGuard g(s);
        tail_kernel<T><<<1, 32, 0, s->stream>>>(tail_args<T>(s), 1);
        CU(cudaGetLastError());
        CU(cudaStreamSynchronize(s->stream));
    }
    return SIM_OK;
}

template <typename T> int slab_step(sim *const *h, int n, int64_t steps)
{
    sim *s0 = h[0];
    SlabCtls t{}; t.n = n;
    for (int r = 0; r < n; ++r) t.c[r] = h[r]->ctl;
    {
        sim *s = s0;
        DeviceGuard g(s);
        int rc = prepare_bins<T>(s);
        if (rc != SIM_OK) return rc;
    }
    Marks none{nullptr, 0, s0->stream};
    for (int64_t k = 0; k < steps; ++k) {
        // fork: the other slabs start after everything of the step before (the binning chain wrote their N_p)
        { sim *s = s0; DeviceGuard g(s); CU(cudaEventRecord(s0->ev_fork, s0->stream)); }
        for (int r = 1; r < n; ++r) { sim *s = h[r]; DeviceGuard g(s); CU(cudaStreamWaitEvent(s->stream, s0->ev_fork, 0)); }
        // pedestrian step (all pedestrians, on the first slab's device) and the flood kernels, all at level n
        {
            sim *s = s0; DeviceGuard g(s);
            if (s->np > 0)
                CU(launch_pdl(ped_step_kernel<T>, dim3((s->np + PED_THREADS - 1) / PED_THREADS), dim3(PED_THREADS), 0, s->stream, false, ped_args_full<T>(s, 0), 0));
        }
        for (int r = 0; r < n; ++r) {
            sim *s = h[r]; DeviceGuard g(s);
            int rc = launch_flood<T>(s, s->stream, false);
            if (rc != SIM_OK) return rc;
            if (r) { CU(cudaEventRecord(s->ev_slab, s->stream)); CU(cudaStreamWaitEvent(s0->stream, s->ev_slab, 0)); }
        }
        // the global wave speed, then every slab's tail
        { sim *s = s0; DeviceGuard g(s); slab_lambda_kernel<<<1, 32, 0, s->stream>>>(t); CU(cudaGetLastError()); CU(cudaEventRecord(s0->ev_ped, s0->stream)); }
        for (int r = 0; r < n; ++r) {
            sim *s = h[r]; DeviceGuard g(s);
            if (r) CU(cudaStreamWaitEvent(s->stream, s0->ev_ped, 0));
            CU(launch_pdl(tail_kernel<T>, dim3(1), dim3(32), 0, s->stream, false, tail_args<T>(s), 0));
            if (r) { CU(cudaEventRecord(s->ev_slab, s->stream)); CU(cudaStreamWaitEvent(s0->stream, s->ev_slab, 0)); }
        }
        // binning chain of the next step (N_p goes to the slab that holds the cell)
        {
            sim *s = s0; DeviceGuard g(s);
            if (s->np > 0) { int rc = enqueue_bin_chain<T>(s, s->stream, 0, none); if (rc != SIM_OK) return rc; }
        }
    }
    return SIM_OK;
}

}  // namespace

extern "C" int sim_slab_link(sim_t *const *h, int32_t n)
{
    if (!h || n < 1 || n > MAX_SLABS) return fail(nullptr, SIM_EINVAL, "1..8 slab handles");
    sim *s = h[0];
    if (!s) return SIM_EINVAL;
    int row = 0;
    for (int r = 0; r < n; ++r) {
        sim *q = h[r];
        if (!q) return fail(s, SIM_EINVAL, "null slab handle");
        if (q->grid.nx != s->grid.nx || q->gny != s->gny || q->grid.real_bits != s->grid.real_bits || q->grid.dx != s->grid.dx || q->grid.dy != s->grid.dy)
            return fail(s, SIM_EINVAL, "slabs must cut one grid");
        if (q->j0 != row) return fail(s, SIM_EINVAL, "slabs must be given in row order and cover the grid without gaps");
        if (r + 1 < n && q->grid.ny != s->grid.ny) return fail(s, SIM_EINVAL, "all slabs but the last must have the same number of rows");
        if (r > 0 && q->np > 0) return fail(s, SIM_EINVAL, "all pedestrians live on the first slab's handle");
        if (q->prm.open_sides || q->prm.flood_order == 2) return fail(s, SIM_EINVAL, "row slabs are not combined with open edges or flood_order 2");
        if (q->ngroup) return fail(s, SIM_EINVAL, "handle is already linked");
        row += q->grid.ny;
    }
    if (row != s->gny) return fail(s, SIM_EINVAL, "slabs must cover the grid");
    // peer access between the devices of the slabs (one process)
    for (int a = 0; a < n; ++a)
        for (int b = 0; b < n; ++b) {
            if (h[a]->device == h[b]->device) continue;
            int can = 0;
            DeviceGuard g(h[a]);
            if (cudaDeviceCanAccessPeer(&can, h[a]->device, h[b]->device) != cudaSuccess || !can)
                return fail(s, SIM_ECUDA, "the devices of the slabs have no peer access");
            cudaError_t e = cudaDeviceEnablePeerAccess(h[b]->device, 0);
            if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) return fail(s, SIM_ECUDA, cudaGetErrorString(e));
            cudaGetLastError();
        }
    for (int r = 0; r < n; ++r) {
        sim *q = h[r];
        DeviceGuard g(q);
        CU(cudaStreamSynchronize(q->stream));
        drop_graphs(q);
        q->ngroup = n; q->grank = r;
        for (int k = 0; k < n; ++k) {
            q->group[k] = h[k];
            sim::Peer &pr = q->peer[k];
            pr.j0 = h[k]->j0; pr.ny = h[k]->grid.ny; pr.zs = h[k]->zs; pr.occ = h[k]->occ; pr.ctl = h[k]->ctl;
            for (int b = 0; b < 2; ++b) { pr.h[b] = h[k]->h[b]; pr.qx[b] = h[k]->qx[b]; pr.qy[b] = h[k]->qy[b]; }
        }
        // the halo row is read by the TMA path of variant 4 (strips inside the domain) and by variant 0
        q->flood_variant = q->grid.nx % MW == 0 && q->flood_variant != 0 ? 4 : 0;
        CU(cudaMemsetAsync(q->dryseg, 0, 2 * q->dry_stride, q->stream));
        if (!q->ev_slab) CU(cudaEventCreateWithFlags(&q->ev_slab, cudaEventDisableTiming));
        q->binned = false;
    }
    return s->grid.real_bits == 64 ? slab_refresh<double>(h, n) : slab_refresh<float>(h, n);
}

extern "C" int sim_slab_describe(sim_t *s, sim_slab_desc_t *o)
{
    if (!s || !o) return SIM_EINVAL;
    std::memset(o, 0, sizeof *o);
    o->j0 = s->j0; o->ny = s->grid.ny;
    for (int k = 0; k < 2; ++k) { o->h[k] = (uint64_t)(uintptr_t)s->h[k]; o->qx[k] = (uint64_t)(uintptr_t)s->qx[k]; o->qy[k] = (uint64_t)(uintptr_t)s->qy[k]; }
    o->zs = (uint64_t)(uintptr_t)s->zs; o->occ = (uint64_t)(uintptr_t)s->occ; o->ctl = (uint64_t)(uintptr_t)s->ctl;
    o->lam_bits = (uint64_t)(uintptr_t)&s->ctl->lam_bits;
    o->workspace = (uint64_t)(uintptr_t)s->ws; o->workspace_bytes = (uint64_t)s->ws_bytes;
    return SIM_OK;
}

extern "C" int sim_slab_attach(sim_t *s, int32_t rank, int32_t n, const sim_slab_desc_t *d)
{
    if (!s || !d || n < 1 || n > MAX_SLABS || rank < 0 || rank >= n) return SIM_EINVAL;
    DeviceGuard on_device(s);
    if (s->ngroup) return fail(s, SIM_EINVAL, "handle is already linked");
    if (s->prm.open_sides || s->prm.flood_order == 2 || s->prm.n_doors > 0)
        return fail(s, SIM_EINVAL, "row slabs over processes are not combined with open edges, flood_order 2 or doors");
    int row = 0;
    for (int r = 0; r < n; ++r) {
        if (d[r].j0 != row || d[r].ny <= 0) return fail(s, SIM_EINVAL, "slabs must be given in row order and cover the grid without gaps");
        if (r + 1 < n && d[r].ny != d[0].ny) return fail(s, SIM_EINVAL, "all slabs but the last must have the same number of rows");
        row += d[r].ny;
    }
    if (row != s->gny || d[rank].j0 != s->j0 || d[rank].ny != s->grid.ny) return fail(s, SIM_EINVAL, "the descriptions do not match this handle's grid");
    if (rank > 0 && s->np > 0) return fail(s, SIM_EINVAL, "all pedestrians live on the first slab's handle");
    // A sandbag deposit raises the bed from the FIRST slab's tail kernel (the pedestrians live there).  Into
    // another process's rows that write is not ordered against that process's next flood kernel: the one
    // exchange of the step, the wave-speed all-reduce, comes before the tails.  So the line must lie in
    // the first slab's rows (sim_slab_link, one process and one host thread launching everything, has no such limit).
    if (n > 1 && s->n_line > 0 && s->line_row_max >= d[0].ny)
        return fail(s, SIM_EINVAL, "row slabs over processes: every barrier cell must lie in the first slab's rows");
    CU(cudaStreamSynchronize(s->stream));
    drop_graphs(s);
    for (int r = 0; r < n; ++r) {
        sim::Peer &pr = s->peer[r];
        pr.j0 = d[r].j0; pr.ny = d[r].ny; pr.zs = (void *)(uintptr_t)d[r].zs; pr.occ = (uint8_t *)(uintptr_t)d[r].occ; pr.ctl = (Ctl *)(uintptr_t)d[r].ctl;
        for (int b = 0; b < 2; ++b) { pr.h[b] = (void *)(uintptr_t)d[r].h[b]; pr.qx[b] = (void *)(uintptr_t)d[r].qx[b]; pr.qy[b] = (void *)(uintptr_t)d[r].qy[b]; }
        s->group[r] = nullptr;
    }
    s->group[rank] = s;
    s->ngroup = n; s->grank = rank;
    s->flood_variant = s->grid.nx % MW == 0 && s->flood_variant != 0 ? 4 : 0;   // see sim_slab_link
    CU(cudaMemsetAsync(s->dryseg, 0, 2 * s->dry_stride, s->stream));
    s->binned = false;
    return SIM_OK;
}

namespace {
template <typename T> int slab_enqueue(sim *s, int phase)
{
    Marks none{nullptr, 0, s->stream};
    if (phase == 0) {
        if (s->np > 0) {
            // The bins (and the N_p they put into the OTHER processes' slabs) must be in place before any
            // rank's flood kernel of this step starts: only phase 2 has the all-reduce between it and them.
            if (!s->binned) return fail(s, SIM_EINVAL, "pedestrians or modes changed since the bins were made: run phase 2, the all-reduce and phase 3 again (binding.SlabRank.resync)");
            int rc = SIM_OK;
            // pedestrian step n with the count of the next chain folded in, then that chain (it fills the N_p
            // buffer the flood kernels of step n are not reading, in whichever slab holds the cell)
            CU(launch_pdl(ped_step_kernel<T>, dim3((s->np + PED_THREADS - 1) / PED_THREADS), dim3(PED_THREADS), 0, s->stream, false, ped_args_full<T>(s, 0), 1));
            rc = enqueue_bin_chain<T>(s, s->stream, 1, none, true);
            if (rc != SIM_OK) return rc;
        }
        return launch_flood<T>(s, s->stream, false);
    }
    if (phase == 1) { CU(launch_pdl(tail_kernel<T>, dim3(1), dim3(32), 0, s->stream, false, tail_args<T>(s), 0)); return SIM_OK; }
    if (phase == 2) {
        if (s->np > 0) {                               // binning chain of the first step: its N_p lands in every slab before the all-reduce
            s->binned = false;
            int rc = prepare_bins<T>(s);
            if (rc != SIM_OK) return rc;
        }
        flood_chunk_flags_kernel<T><<<dim3(s->march_gx, s->march_gy), 256, 0, s->stream>>>((const T *)s->zs, s->grid.nx, s->grid.ny, s->march_R, s->chunk_flag);
        flood_lambda_kernel<T><<<592, 256, 0, s->stream>>>(flood_args<T>(s));
        CU(cudaGetLastError());
        return SIM_OK;
    }
    if (phase == 3) { tail_kernel<T><<<1, 32, 0, s->stream>>>(tail_args<T>(s), 1); CU(cudaGetLastError()); return SIM_OK; }
    return fail(s, SIM_EINVAL, "phase must be 0..3");
}
}  // namespace

extern "C" int sim_slab_enqueue(sim_t *s, int32_t phase)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    if (s->ngroup < 1 || s->group[s->grank] != s) return fail(s, SIM_EINVAL, "sim_slab_attach first");
    return DISPATCH(s, slab_enqueue, s, phase);
}

extern "C" int sim_slab_step(sim_t *const *h, int32_t n, int64_t steps)
{
    if (!h || n < 1 || !h[0]) return SIM_EINVAL;
    sim *s = h[0];
    if (s->ngroup != n) return fail(s, SIM_EINVAL, "sim_slab_link these handles first");
    for (int r = 0; r < n; ++r) if (h[r] != s->group[r]) return fail(s, SIM_EINVAL, "not the linked handles, or not in their order");
    if (steps < 0) return fail(s, SIM_EINVAL, "negative step count");
    return s->grid.real_bits == 64 ? slab_step<double>(h, n, steps) : slab_step<float>(h, n, steps);
}

extern "C" int sim_test_philox(sim_t *s, const uint32_t *in, uint32_t *out, int32_t n)
{
    if (!s || !in || !out || n < 0) return SIM_EINVAL;
    DeviceGuard on_device(s);
    if (n == 0) return SIM_OK;
    unsigned *d = nullptr;
    CU(cudaMalloc(&d, (size_t)n * 10 * sizeof(unsigned)));
    struct Free { unsigned *p; ~Free() { cudaFree(p); } } fr{d};
    CU(cudaMemcpyAsync(d, in, (size_t)n * 6 * sizeof(unsigned), cudaMemcpyHostToDevice, s->stream));
    philox_test_kernel<<<(n + 127) / 128, 128, 0, s->stream>>>(d, d + (size_t)n * 6, n);
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(out, d + (size_t)n * 6, (size_t)n * 4 * sizeof(unsigned), cudaMemcpyDeviceToHost, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    return SIM_OK;
}

extern "C" int sim_get_flood_variant(const sim_t *s) { return s ? s->flood_variant : SIM_EINVAL; }

extern "C" int sim_set_flood_variant(sim_t *s, int32_t variant)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    if (variant < 0 || variant > 4) return fail(s, SIM_EINVAL, "variant must be 0..4");
    if (s->prm.flood_order == 2) return fail(s, SIM_EINVAL, "flood_order = 2 has one kernel (variant 5)");
    if (s->prm.open_sides && variant != 0) return fail(s, SIM_EINVAL, "open edges are built into variants 0 and 5 only");
    if (s->ngroup > 1 && !(variant == 0 || (variant == 4 && s->grid.nx % MW == 0)))
        return fail(s, SIM_EINVAL, "a linked row slab runs variant 0, or variant 4 when nx is a multiple of 256 (the halo row is read by those)");
    if (variant == 4 && s->grid.nx % 16 != 0) return fail(s, SIM_EINVAL, "the TMA march kernel needs nx % 16 == 0");
    if (variant == 3 && s->grid.nx % 2 != 0) return fail(s, SIM_EINVAL, "the two-column march kernel needs nx % 2 == 0");
    if (variant == 1 && s->grid.nx % 4 != 0) return fail(s, SIM_EINVAL, "the tiled kernel needs nx % 4 == 0");
    CU(cudaStreamSynchronize(s->stream));
    s->flood_variant = variant;
    drop_graphs(s);
    CU(cudaMemsetAsync(s->dryseg, 0, 2 * s->dry_stride, s->stream));       // only the TMA march kernel keeps the dry flags up to date
    return SIM_OK;
}

extern "C" int sim_set_dry_skip(sim_t *s, int32_t on)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    CU(cudaStreamSynchronize(s->stream));
    s->dry_skip = on ? 1 : 0;
    drop_graphs(s);
    CU(cudaMemsetAsync(s->dryseg, 0, 2 * s->dry_stride, s->stream));
    return SIM_OK;
}

extern "C" int sim_set_deterministic(sim_t *s, int32_t on)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    CU(cudaStreamSynchronize(s->stream));
    s->deterministic = on ? 1 : 0;
    s->binned = false;                     // the bins in place were ordered the other way: sort again before the next step
    drop_graphs(s);
    return SIM_OK;
}

namespace {

template <typename T> int read_flood_t(sim *s, void *h, void *u, void *v, void *z, void *hr)
{
    const size_t bytes = (size_t)s->ncell * sizeof(T);
    Ctl c;
    CU(cudaMemcpyAsync(&c, s->ctl, sizeof c, cudaMemcpyDeviceToHost, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    if (u || v || hr) {
        flood_derive_kernel<T><<<1184, 256, 0, s->stream>>>(flood_args<T>(s), u ? (T *)s->scratch_real[0] : nullptr,
                                                          v ? (T *)s->scratch_real[1] : nullptr,
                                                          hr ? (T *)s->scratch_real[2] : nullptr);
        CU(cudaGetLastError());
    }
    if (copy_out(s, h, s->h[c.parity], bytes) || copy_out(s, u, s->scratch_real[0], bytes) ||
        copy_out(s, v, s->scratch_real[1], bytes) || copy_out(s, hr, s->scratch_real[2], bytes))
        return SIM_ECUDA;
    if (z) {
        // bed with the barrier raised; solid cells report the elevation they were created with
        flood_bed_kernel<T><<<1184, 256, 0, s->stream>>>((const T *)s->zs, (const T *)s->z0, (size_t)s->ncell, (T *)s->scratch_real[0]);
        CU(cudaGetLastError());
        if (copy_out(s, z, s->scratch_real[0], bytes)) return SIM_ECUDA;
    }
    CU(cudaStreamSynchronize(s->stream));
    return SIM_OK;
}

template <typename T> int read_peds_t(sim *s, void *x, void *y, void *vx, void *vy, uint8_t *state, uint8_t *fsm,
                                      uint8_t *active, int32_t *cell, void *timer)
{
    const int np = s->np;
    if (!np) return SIM_OK;
    ped_gather_kernel<T><<<(np + 255) / 256, 256, 0, s->stream>>>(
        ped_soa<T>(s, 0), np, s->grid.nx, (T)(1.0 / s->grid.dx), (T)(1.0 / s->grid.dy), s->gny,
        (T *)s->ped_out[0], (T *)s->ped_out[1], (T *)s->ped_out[2], (T *)s->ped_out[3],
        s->ped_out_u8[0], s->ped_out_u8[1], s->ped_out_u8[2], s->ped_out_i32[0], (T *)s->ped_out[4], nullptr);
    CU(cudaGetLastError());
    const size_t rb = (size_t)np * sizeof(T);
    if (copy_out(s, x, s->ped_out[0], rb) || copy_out(s, y, s->ped_out[1], rb) || copy_out(s, vx, s->ped_out[2], rb) ||
        copy_out(s, vy, s->ped_out[3], rb) || copy_out(s, timer, s->ped_out[4], rb) ||
        copy_out(s, state, s->ped_out_u8[0], np) || copy_out(s, fsm, s->ped_out_u8[1], np) ||
        copy_out(s, active, s->ped_out_u8[2], np) || copy_out(s, cell, s->ped_out_i32[0], (size_t)np * 4))
        return SIM_ECUDA;
    CU(cudaStreamSynchronize(s->stream));
    return SIM_OK;
}

template <typename T> int stats_t(sim *s, sim_stats_t *o)
{
    CU(cudaMemsetAsync(s->stat_d, 0, 8 * sizeof(double), s->stream));
    CU(cudaMemsetAsync(s->stat_hist, 0, 8 * sizeof(unsigned long long), s->stream));
    flood_stats_kernel<T><<<1184, 256, 0, s->stream>>>(flood_args<T>(s), s->stat_d);
    if (s->np) ped_hist_kernel<T><<<(s->np + 255) / 256, 256, 0, s->stream>>>(ped_soa<T>(s, 0), s->np, s->stat_hist, s->stat_d + 4);
    CU(cudaGetLastError());
    double d[8]; unsigned long long hist[8]; Ctl c;
    CU(cudaMemcpyAsync(d, s->stat_d, sizeof d, cudaMemcpyDeviceToHost, s->stream));
    CU(cudaMemcpyAsync(hist, s->stat_hist, sizeof hist, cudaMemcpyDeviceToHost, s->stream));
    CU(cudaMemcpyAsync(&c, s->ctl, sizeof c, cudaMemcpyDeviceToHost, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    std::memset(o, 0, sizeof *o);
    o->t = c.t; o->dt = c.dt; o->step = c.step;
    o->volume = d[0]; o->max_h = d[1]; o->max_hr = d[2];
    for (int k = 0; k < 6; ++k) o->hist[k] = (int64_t)hist[k];
    o->neg_depth_clamps = (int64_t)c.neg_clamps; o->clamped_volume = c.clamped_volume;
    o->cursor = c.cursor; o->layer = c.layer; o->bags = c.bags; o->barrier_complete = c.complete;
    o->deposits = c.deposits;
    o->outflow_volume = c.outflow_volume; o->spawned = c.spawned; o->triggered = c.triggered;
    if (d[3] > 0 || d[4] > 0) return fail(s, SIM_ENOTFINITE, "non-finite depth, discharge or position");
    return SIM_OK;
}

template <typename T> int bin_peds_t(sim *s, int32_t *key, int32_t *order, int32_t *start)
{
    const int np = s->np;
    if (np) {
        PedArgs<T> pa = ped_args<T>(s);
        const int nb = (np + 255) / 256, n_items = s->nbins + 1;
        Ctl c;
        CU(cudaMemcpyAsync(&c, s->ctl, sizeof c, cudaMemcpyDeviceToHost, s->stream));
        CU(cudaStreamSynchronize(s->stream));
        const int halt = c.halt;
        if (halt) { c.halt = 0; CU(cudaMemcpyAsync(s->ctl, &c, sizeof c, cudaMemcpyHostToDevice, s->stream)); }
        ped_bin_count_kernel<T><<<nb, 256, 0, s->stream>>>(pa, 0);
        scan_bins_kernel<<<(n_items + SCAN_TILE - 1) / SCAN_TILE, SCAN_THREADS, 0, s->stream>>>(s->count, s->start, n_items, s->scan_status, s->ctl, 0, 0);
        if (s->deterministic) { ped_perm_kernel<T><<<nb, 256, 0, s->stream>>>(pa); ped_rank_kernel<T><<<nb, 256, 0, s->stream>>>(pa); }
        ped_scatter_kernel<T><<<nb, 256, 0, s->stream>>>(pa);
        ped_key_by_id_kernel<T><<<nb, 256, 0, s->stream>>>(ped_soa<T>(s, 0), s->key, np, s->ped_out_i32[0]);
        ped_gather_kernel<T><<<nb, 256, 0, s->stream>>>(ped_soa<T>(s, 1), np, s->grid.nx, (T)1, (T)1, s->gny,
            nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, s->ped_out_i32[1]);
        CU(cudaGetLastError());
        // (the scatter kernel has re-armed the scan)
        CU(cudaMemcpyAsync(&c, s->ctl, sizeof c, cudaMemcpyDeviceToHost, s->stream));
        CU(cudaStreamSynchronize(s->stream));
        c.halt = halt;
        s->binned = false;
        CU(cudaMemcpyAsync(s->ctl, &c, sizeof c, cudaMemcpyHostToDevice, s->stream));
        if (copy_out(s, key, s->ped_out_i32[0], (size_t)np * 4) || copy_out(s, order, s->ped_out_i32[1], (size_t)np * 4))
            return SIM_ECUDA;
    }
    if (np == 0) CU(cudaMemsetAsync(s->start, 0, (size_t)(s->nbins + 2) * 4, s->stream));
    if (copy_out(s, start, s->start, (size_t)(s->nbins + 2) * 4)) return SIM_ECUDA;
    CU(cudaStreamSynchronize(s->stream));
    return SIM_OK;
}

template <typename T> int write_flood_t(sim *s, const void *h, const void *qx, const void *qy, const void *z)
{
    const size_t nc = (size_t)s->ncell, bytes = nc * sizeof(T);
    Ctl c;
    CU(cudaMemcpyAsync(&c, s->ctl, sizeof c, cudaMemcpyDeviceToHost, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    const int p = c.parity;
    if (h) CU(cudaMemcpyAsync(s->h[p], h, bytes, cudaMemcpyHostToDevice, s->stream));
    if (qx) CU(cudaMemcpyAsync(s->qx[p], qx, bytes, cudaMemcpyHostToDevice, s->stream));
    if (qy) CU(cudaMemcpyAsync(s->qy[p], qy, bytes, cudaMemcpyHostToDevice, s->stream));
    if (z) CU(cudaMemcpyAsync(s->scratch_real[0], z, bytes, cudaMemcpyHostToDevice, s->stream));
    // solid cells hold no water and keep z = +inf; then the CFL dt, q_in and halt of the injected state
    CU(cudaMemsetAsync(s->dryseg, 0, 2 * s->dry_stride, s->stream));       // state written from outside: nothing is known to be dry
    flood_inject_kernel<T><<<1184, 256, 0, s->stream>>>((T *)s->h[p], (T *)s->qx[p], (T *)s->qy[p], (T *)s->zs,
                                                       z ? (const T *)s->scratch_real[0] : nullptr, nc);
    CU(cudaGetLastError());
    int rc = refresh_dt<T>(s);
    if (rc != SIM_OK) return rc;
    CU(cudaStreamSynchronize(s->stream));
    return SIM_OK;
}

}  // namespace

extern "C" int sim_read_flood(sim_t *s, void *h, void *u, void *v, void *z, void *hr)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    return DISPATCH(s, read_flood_t, s, h, u, v, z, hr);
}

extern "C" int sim_read_conserved(sim_t *s, void *h, void *qx, void *qy)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    Ctl c;
    CU(cudaMemcpyAsync(&c, s->ctl, sizeof c, cudaMemcpyDeviceToHost, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    const size_t bytes = (size_t)s->ncell * real_size(s);
    if (copy_out(s, h, s->h[c.parity], bytes) || copy_out(s, qx, s->qx[c.parity], bytes) ||
        copy_out(s, qy, s->qy[c.parity], bytes)) return SIM_ECUDA;
    CU(cudaStreamSynchronize(s->stream));
    return SIM_OK;
}

extern "C" int sim_read_occupancy(sim_t *s, uint8_t *np_cell)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    Ctl c;
    CU(cudaMemcpyAsync(&c, s->ctl, sizeof c, cudaMemcpyDeviceToHost, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    // the most recent step ran at flood parity c.parity ^ 1 and read that N_p buffer
    if (copy_out(s, np_cell, s->occ + (size_t)(c.parity ^ 1) * s->ncell, (size_t)s->ncell)) return SIM_ECUDA;
    CU(cudaStreamSynchronize(s->stream));
    return SIM_OK;
}

extern "C" int sim_read_peds(sim_t *s, void *x, void *y, void *vx, void *vy, uint8_t *state, uint8_t *fsm,
                             uint8_t *active, int32_t *cell, void *timer)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    return DISPATCH(s, read_peds_t, s, x, y, vx, vy, state, fsm, active, cell, timer);
}

extern "C" int sim_get_stats(sim_t *s, sim_stats_t *out)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    if (!out) return fail(s, SIM_EINVAL, "out is NULL");
    return DISPATCH(s, stats_t, s, out);
}

extern "C" int sim_bin_peds(sim_t *s, int32_t *key, int32_t *order, int32_t *start,
                            int32_t *n_bins_x, int32_t *n_bins_y, int32_t *k)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    if (n_bins_x) *n_bins_x = s->nbx;
    if (n_bins_y) *n_bins_y = s->nby;
    if (k) *k = s->kbin;
    if (!key && !order && !start) return SIM_OK;
    return DISPATCH(s, bin_peds_t, s, key, order, start);
}

extern "C" int sim_write_flood(sim_t *s, const void *h, const void *qx, const void *qy, const void *z)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    s->binned = false;
    return DISPATCH(s, write_flood_t, s, h, qx, qy, z);
}

extern "C" int sim_write_peds(sim_t *s, const void *x, const void *y, const void *vx, const void *vy,
                              const uint8_t *fsm, const uint8_t *active, const void *timer)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    s->binned = false;
    const size_t np = (size_t)s->np, rb = np * real_size(s);
    if (!np) return SIM_OK;
    // put buffer A back into original order first, so that index i means agent i again
    CU(cudaStreamSynchronize(s->stream));
    int rc = sim_read_peds(s, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr);
    if (rc != SIM_OK) return rc;
    // ped_out_* now hold x y vx vy timer / state fsm active in original order
    auto put = [&](void *dst, const void *host, const void *dev_orig, size_t bytes) -> int {
        if (host) CU(cudaMemcpyAsync(dst, host, bytes, cudaMemcpyHostToDevice, s->stream));
        else CU(cudaMemcpyAsync(dst, dev_orig, bytes, cudaMemcpyDeviceToDevice, s->stream));
        return SIM_OK;
    };
    // vpref / role / id need un-permuting too: do it on the host (test hook, not hot)
    std::vector<int32_t> id(np);
    std::vector<char> vp(rb), vp2(rb);
    std::vector<uint8_t> role(np), role2(np);
    CU(cudaMemcpyAsync(id.data(), s->P[0].id, np * 4, cudaMemcpyDeviceToHost, s->stream));
    CU(cudaMemcpyAsync(vp.data(), s->P[0].vpref, rb, cudaMemcpyDeviceToHost, s->stream));
    CU(cudaMemcpyAsync(role.data(), s->P[0].role, np, cudaMemcpyDeviceToHost, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    const size_t rs = real_size(s);
    for (size_t k = 0; k < np; ++k) { std::memcpy(&vp2[(size_t)id[k] * rs], &vp[k * rs], rs); role2[id[k]] = role[k]; }
    for (size_t k = 0; k < np; ++k) id[k] = (int32_t)k;
    if (put(s->P[0].x, x, s->ped_out[0], rb) || put(s->P[0].y, y, s->ped_out[1], rb) ||
        put(s->P[0].vx, vx, s->ped_out[2], rb) || put(s->P[0].vy, vy, s->ped_out[3], rb) ||
        put(s->P[0].timer, timer, s->ped_out[4], rb) || put(s->P[0].state, nullptr, s->ped_out_u8[0], np) ||
        put(s->P[0].fsm, fsm, s->ped_out_u8[1], np) || put(s->P[0].active, active, s->ped_out_u8[2], np))
        return SIM_ECUDA;
    CU(cudaMemcpyAsync(s->P[0].vpref, vp2.data(), rb, cudaMemcpyHostToDevice, s->stream));
    CU(cudaMemcpyAsync(s->P[0].role, role2.data(), np, cudaMemcpyHostToDevice, s->stream));
    CU(cudaMemcpyAsync(s->P[0].id, id.data(), np * 4, cudaMemcpyHostToDevice, s->stream));
    // occupancy bookkeeping restarts from scratch
    CU(cudaMemsetAsync(s->occ, 0, 2 * (size_t)s->ncell, s->stream));
    CU(cudaMemsetAsync(s->cellprev, 0xff, 2 * np * 4, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    return SIM_OK;
}

extern "C" int sim_set_time(sim_t *s, double t, double dt)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    s->binned = false;
    Ctl c;
    CU(cudaMemcpyAsync(&c, s->ctl, sizeof c, cudaMemcpyDeviceToHost, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    c.t = t; c.dt = dt; c.halt = (t >= c.t_end) ? 1 : 0;
    // same piecewise-linear lookup as the tail kernel, on the host copy of the table
    double q = 0.0;
    const int n = s->n_hydro;
    if (n > 0) {
        std::vector<double> ht(n), hq(n);
        CU(cudaMemcpyAsync(ht.data(), s->hydro_t, (size_t)n * 8, cudaMemcpyDeviceToHost, s->stream));
        CU(cudaMemcpyAsync(hq.data(), s->hydro_q, (size_t)n * 8, cudaMemcpyDeviceToHost, s->stream));
        CU(cudaStreamSynchronize(s->stream));
        if (t <= ht[0]) q = hq[0];
        else { q = hq[n - 1]; for (int k = 0; k + 1 < n; ++k) if (t < ht[k + 1]) { q = hq[k] + (hq[k + 1] - hq[k]) * (t - ht[k]) / (ht[k + 1] - ht[k]); break; } }
    }
    c.q_in = s->inflow_length > 0 ? q / s->inflow_length : 0.0;
    CU(cudaMemcpyAsync(s->ctl, &c, sizeof c, cudaMemcpyHostToDevice, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    return SIM_OK;
}

extern "C" int sim_set_barrier(sim_t *s, int32_t cursor, int32_t layer, int32_t bags, int32_t complete)
{
    if (!s) return SIM_EINVAL;
    DeviceGuard on_device(s);
    s->binned = false;
    Ctl c;
    CU(cudaMemcpyAsync(&c, s->ctl, sizeof c, cudaMemcpyDeviceToHost, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    c.cursor = cursor; c.layer = layer; c.bags = bags; c.complete = complete;
    CU(cudaMemcpyAsync(s->ctl, &c, sizeof c, cudaMemcpyHostToDevice, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    return SIM_OK;
}

extern "C" const char *sim_last_error(const sim_t *s) { return s ? s->err.c_str() : g_create_error.c_str(); }

extern "C" void sim_destroy(sim_t *s)
{
    if (!s) return;
    DeviceGuard on_device(s);
    if (s->ws) cudaStreamSynchronize(s->stream);
    drop_graphs(s);
    if (s->cap_stream) cudaStreamDestroy(s->cap_stream);
    if (s->stream2) cudaStreamDestroy(s->stream2);
    if (s->ev_fork) cudaEventDestroy(s->ev_fork);
    if (s->ev_ped) cudaEventDestroy(s->ev_ped);
    if (s->ev_occ) cudaEventDestroy(s->ev_occ);
    if (s->ev_tail) cudaEventDestroy(s->ev_tail);
    if (s->ev_slab) cudaEventDestroy(s->ev_slab);
    if (s->own_ws && s->ws) cudaFree(s->ws);
    delete s;
}

// ================================================================================ no-allocation entry point
// sim_cfl_dt_static (include/floodped.h): the CFL time step of a flood state the caller holds in device
// memory, for callers that may not allocate device memory at all.  It is a variant of flood_lambda_kernel: the
// per-cell wave speed is the same expression, but where that kernel folds the maximum into the handle's control
// block (part of a workspace somebody allocated), this one keeps its scratch -- a ticket word and one partial
// maximum per block -- in the file-scope array below, which the CUDA module itself carries.  Nothing here calls
// cudaMalloc, cudaFree or a library routine that allocates.
namespace {

constexpr long long CFL_STATIC_MAX_CELLS = SIM_CFL_STATIC_MAX_CELLS;
constexpr int CFL_STATIC_THREADS = 256;
constexpr int CFL_STATIC_BLOCK_CELLS = 8192;                         // 32 cells per thread
constexpr int CFL_STATIC_MAX_BLOCKS = (int)(CFL_STATIC_MAX_CELLS / CFL_STATIC_BLOCK_CELLS);
constexpr int CFL_STATIC_HEAD = 32;                                  // the ticket word has a 256-byte line of its own
static_assert(CFL_STATIC_MAX_CELLS % CFL_STATIC_BLOCK_CELLS == 0, "whole blocks");

// 256 KiB + 256 B per device that loads the library, held until the process exits.  Word 0: how many blocks of
// the running launch have published their partial maximum (must be zero when a launch starts); words
// CFL_STATIC_HEAD + b: partial maximum of block b as the bit pattern of a non-negative double.
// In host code this name is only a handle for cudaGetSymbolAddress -- never pass it to a kernel as it stands.
static __device__ __align__(256) unsigned long long g_cfl_static_scratch[CFL_STATIC_HEAD + CFL_STATIC_MAX_BLOCKS];

template <typename T>
__global__ void __launch_bounds__(CFL_STATIC_THREADS)
cfl_static_kernel(const T *__restrict__ h, const T *__restrict__ qx, const T *__restrict__ qy, const uint8_t *__restrict__ mask,
                  long long n, T g, T h_dry, T inv_dx, T inv_dy, double cfl, double dt_max,
                  unsigned long long *scratch, double *out)
{
    __shared__ T red[32];
    __shared__ unsigned long long redb[32];
    __shared__ int last;
    const int tid = threadIdx.x;
    const long long c0 = (long long)blockIdx.x * CFL_STATIC_BLOCK_CELLS;
    T lam = T(0);
    for (int k = tid; k < CFL_STATIC_BLOCK_CELLS; k += CFL_STATIC_THREADS) {
        const long long c = c0 + k;
        if (c >= n) break;
        const T hh = h[c];
        if (!(mask && mask[c]) && hh > h_dry) {                       // as flood_lambda_kernel (flood.cuh)
            const T u = qx[c] / hh, v = qy[c] / hh, cc = real_sqrt(g * hh);
            lam = fmax(lam, fmax((fabs(u) + cc) * inv_dx, (fabs(v) + cc) * inv_dy));
        }
    }
    for (int o = 16; o > 0; o >>= 1) lam = fmax(lam, __shfl_xor_sync(0xffffffffu, lam, o));
    if ((tid & 31) == 0) red[tid >> 5] = lam;
    __syncthreads();
    if (tid < 32) {
        T m = tid < CFL_STATIC_THREADS / 32 ? red[tid] : T(0);
        for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (tid == 0) {
            scratch[CFL_STATIC_HEAD + blockIdx.x] = (unsigned long long)__double_as_longlong((double)m);
            __threadfence();                                          // the partial is visible before the ticket counts it
            last = atomicAdd(&scratch[0], 1ull) == (unsigned long long)gridDim.x - 1ull;
        }
    }
    __syncthreads();
    if (!last) return;
    // the block that took the last ticket folds the partials: max over bit patterns of non-negative doubles
    __threadfence();
    unsigned long long m = 0ull;
    const volatile unsigned long long *part = scratch + CFL_STATIC_HEAD;
    for (unsigned b = tid; b < gridDim.x; b += CFL_STATIC_THREADS) { const unsigned long long v = part[b]; m = v > m ? v : m; }
    for (int o = 16; o > 0; o >>= 1) { const unsigned long long v = __shfl_xor_sync(0xffffffffu, m, o); m = v > m ? v : m; }
    if ((tid & 31) == 0) redb[tid >> 5] = m;
    __syncthreads();
    if (tid == 0) {
        for (int w = 1; w < CFL_STATIC_THREADS / 32; ++w) m = redb[w] > m ? redb[w] : m;
        const double lmax = __longlong_as_double((long long)m);
        double dt = dt_max;                                           // as tail_kernel (peds.cuh), without its t_end clamp
        if (lmax > 0.0) dt = fmin(dt, cfl / lmax);
        out[0] = lmax; out[1] = dt;
        scratch[0] = 0ull;                                            // ready for the next launch
    }
}

// Device address of the scratch array on `dev`, looked up once per device with that device current.
int cfl_static_scratch(int dev, unsigned long long **out)
{
    sim *s = nullptr;                                                 // CU(): errors go to sim_last_error(NULL)
    constexpr int MAXDEV = 64;
    static unsigned long long *addr[MAXDEV] = {};
    static std::mutex mu;
    std::lock_guard<std::mutex> lock(mu);
    if (dev >= 0 && dev < MAXDEV && addr[dev]) { *out = addr[dev]; return SIM_OK; }
    int cur = -1;
    CU(cudaGetDevice(&cur));
    if (cur != dev) CU(cudaSetDevice(dev));
    unsigned long long *p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void **)&p, g_cfl_static_scratch);
    if (cur != dev) cudaSetDevice(cur);
    if (e != cudaSuccess || !p)
        return fail(nullptr, SIM_ECUDA, std::string("cudaGetSymbolAddress(g_cfl_static_scratch): ") + cudaGetErrorString(e));
    if (dev >= 0 && dev < MAXDEV) addr[dev] = p;
    *out = p;
    return SIM_OK;
}

}  // namespace

extern "C" int sim_cfl_dt_static(const void *h, const void *qx, const void *qy, const uint8_t *mask, int64_t n_cells,
                                 int32_t real_bits, double dx, double dy, double g, double h_dry, double cfl,
                                 double dt_max, void *cuda_stream, double *out)
{
    sim *s = nullptr;
    if (n_cells < 0) return fail(nullptr, SIM_EINVAL, "sim_cfl_dt_static: negative n_cells");
    if (n_cells > CFL_STATIC_MAX_CELLS)
        return fail(nullptr, SIM_EINVAL, "sim_cfl_dt_static: n_cells = " + std::to_string((long long)n_cells) +
                    " is beyond SIM_CFL_STATIC_MAX_CELLS = " + std::to_string(CFL_STATIC_MAX_CELLS) +
                    " (the scratch of this entry point is a fixed array; use sim_create with a workspace for larger grids)");
    if (!out || (n_cells > 0 && (!h || !qx || !qy))) return fail(nullptr, SIM_EINVAL, "sim_cfl_dt_static: h, qx, qy and out are required");
    if (real_bits != 32 && real_bits != 64) return fail(nullptr, SIM_EINVAL, "sim_cfl_dt_static: real_bits must be 32 or 64");
    if (!(dx > 0) || !(dy > 0) || !(g > 0) || !(cfl > 0) || !(h_dry > 0) || !(dt_max > 0))
        return fail(nullptr, SIM_EINVAL, "sim_cfl_dt_static: dx, dy, g, cfl, h_dry and dt_max must be positive");
    int dev = -1;
    CU(cudaGetDevice(&dev));
    unsigned long long *scratch = nullptr;
    int rc = cfl_static_scratch(dev, &scratch);
    if (rc != SIM_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int blocks = n_cells > 0 ? (int)((n_cells + CFL_STATIC_BLOCK_CELLS - 1) / CFL_STATIC_BLOCK_CELLS) : 1;
    // the ticket must start at zero whatever the launch before left behind (e.g. one that was aborted)
    CU(cudaMemsetAsync(scratch, 0, sizeof(unsigned long long), st));
    if (real_bits == 64)
        cfl_static_kernel<double><<<blocks, CFL_STATIC_THREADS, 0, st>>>((const double *)h, (const double *)qx, (const double *)qy, mask,
            (long long)n_cells, g, h_dry, 1.0 / dx, 1.0 / dy, cfl, dt_max, scratch, out);
    else
        cfl_static_kernel<float><<<blocks, CFL_STATIC_THREADS, 0, st>>>((const float *)h, (const float *)qx, (const float *)qy, mask,
            (long long)n_cells, (float)g, (float)h_dry, (float)(1.0 / dx), (float)(1.0 / dy), cfl, dt_max, scratch, out);
    CU(cudaGetLastError());
    return SIM_OK;
}
