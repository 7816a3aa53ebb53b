/*
 * floodped.h -- C ABI of libfloodped.so: the coupled flood-pedestrian timestep of
 * Shirvani, Kesserwani & Richmond, "Agent-based simulator of dynamic flood-people
 * interactions" (arXiv 1908.05232), hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * Citations: "P:L<n>" = line n of the paper text; "C<nn>" = the reading of
 * that number in DESIGN.md section 3 (where the paper is silent, ambiguous or garbled).
 *
 * One coupled step n -> n+1, every read at level n (the paper's simultaneous update of
 * all agents):
 *   (O) pedestrians per cell N_p -> roughness n = n0 (1 + min(N_p, n_cap))
 *   (F) flood cells: first-order finite-volume update of U = [h, hu, hv], Eq. (2),
 *       Riemann fluxes on hydrostatically reconstructed states, Manning friction
 *       (sim_params_t::flood_order = 2: the second-order scheme it was reduced from)
 *   (T) t += dt ; dt for the next step from the CFL criterion, on the device
 *   (B) pedestrians binned by counting sort + prefix scan (replaces FLAMEGPU's
 *       per-cell messages)
 *   (P) pedestrian step: HR = (V + 0.5) h -> Table 1 state and speed, navigation,
 *       social force over adjacent bins, move, responder actions, exit
 *   (S) sandbags dropped this step raise the bed z of the barrier line
 *
 * Conventions
 *  - Every function returns SIM_OK (0) or a negative SIM_E* code; nothing throws or aborts
 *    across this boundary.  sim_last_error() gives a human-readable reason.
 *  - Grid arrays are row-major [j][i], ny rows of nx cells; cell (i,j) has centre
 *    ((i+.5)dx, (j+.5)dy); a cell index is j*nx+i.
 *  - "real" arrays hold float when grid.real_bits == 32 and double when it is 64; that is
 *    also the precision the kernels compute in.
 *  - INPUT pointers of sim_create / sim_write_* are HOST pointers, borrowed for the call and
 *    copied.  OUTPUT pointers of sim_read_* may be HOST or DEVICE pointers (detected with
 *    cudaPointerGetAttributes); the caller owns them and they must hold the stated length.
 *  - If `workspace` is non-NULL it is a DEVICE buffer of at least sim_workspace_bytes()
 *    bytes (e.g. a torch.empty uint8 tensor) that holds ALL device state; the library then
 *    never calls cudaMalloc and the caller frees the buffer after sim_destroy.
 *  - `cuda_stream` is a cudaStream_t (NULL = legacy default stream).  sim_step only enqueues
 *    work on it and never synchronises; sim_read_*, sim_get_stats synchronise it.
 *  - A handle is not thread-safe; distinct handles are independent.
 *  - There is no CPU fallback: without a CUDA device sim_create fails with SIM_ECUDA.
 */
#ifndef FLOODPED_H
#define FLOODPED_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SIM_OK          0
#define SIM_EINVAL     -1   /* bad argument (which one: sim_last_error)          */
#define SIM_ENOMEM     -2   /* workspace too small or device allocation failed   */
#define SIM_ECUDA      -3   /* CUDA runtime error, or no device                  */
#define SIM_ENOTFINITE -4   /* a non-finite depth or position was found at read  */

/* cell sides for inflow faces */
#define SIM_SIDE_W 0
#define SIM_SIDE_E 1
#define SIM_SIDE_S 2
#define SIM_SIDE_N 3
/* flood-risk state of a pedestrian: Table 1 plus "dry" (C17) */
#define SIM_STATE_DRY 0
#define SIM_STATE_LOW 1
#define SIM_STATE_MEDIUM 2
#define SIM_STATE_HIGH 3
#define SIM_STATE_HIGHEST 4
/* responder finite-state machine; evacuees are always SIM_FSM_EVACUATE */
#define SIM_FSM_EVACUATE 0
#define SIM_FSM_TO_STORAGE 1
#define SIM_FSM_PICKING 2
#define SIM_FSM_TO_BARRIER 3
#define SIM_FSM_DROPPING 4
/* entered through a door before the flood and walking to destination door d: SIM_FSM_WANDER + d
 * (P:L164, L186); becomes SIM_FSM_EVACUATE at the trigger */
#define SIM_FSM_WANDER 8
/* navigation direction codes: 0..7 = E,NE,N,NW,W,SW,S,SE */
#define SIM_DIR_NONE 255

typedef struct sim sim_t;                       /* opaque, owned by the library */

typedef struct {
    int32_t nx, ny;
    double  dx, dy;                             /* cell size, m                  */
    int32_t real_bits;                          /* 32 or 64                               */
    /* Row slab (both 0 = the whole grid).  This handle holds the flood cells of rows
     * [slab_j0, slab_j0 + ny) of a grid of slab_ny_global rows.  Every array given to sim_create
     * (z, mask, h0, u0, v0, manning, nav_dir) is then the array of the WHOLE grid, every cell index
     * (inflow, exit, door, barrier cells) is a cell of the whole grid, and the handle takes what it
     * needs.  sim_read_* / sim_write_flood move the slab's rows only.  See sim_slab_link(). */
    int32_t slab_j0, slab_ny_global;
} sim_grid_t;

typedef struct {                                /* flood agents' initial state    */
    const void    *z;                           /* [ny*nx] real, bed elevation            */
    const uint8_t *mask;                        /* [ny*nx] 1 = solid/impassable; NULL = none (C16) */
    const void    *h0, *u0, *v0;                /* [ny*nx] real; NULL = 0                 */
} sim_topo_t;

typedef struct {                                /* pedestrian agents        */
    int32_t        n;
    const void    *x, *y, *vx, *vy, *v_pref;    /* [n] real; v_pref = dry walking speed */
    const uint8_t *role;                        /* [n] 0 evacuee, 1 responder             */
    const uint8_t *active;                      /* [n] 1 = in the domain at t = 0; NULL = everybody.  Inactive slots are
                                                   free for newcomers   */
} sim_peds_t;

typedef struct {
    /* hydrodynamics */
    double  g, cfl, dt_max, h_dry;              /* 9.81, 0.5, <=0 => C10 default, 1e-3 (C5, C7, C9) */
    int32_t couple_roughness, n_cap;            /* people -> roughness on/off; cap 20; n_cap <= 255 */
    /* inflow (C14): faces on the domain edge, wall for momentum, mass flux Q(t)/length */
    int32_t        n_inflow_faces;
    const int32_t *inflow_cell;                 /* [n_inflow_faces] cell index on the edge named by side */
    const uint8_t *inflow_side;                 /* [n_inflow_faces] SIM_SIDE_*            */
    int32_t        n_hydro;
    const double  *hydro_t, *hydro_q;           /* [n_hydro] piecewise-linear Q(t), m3/s, t increasing */
    /* Table 1 */
    double  hr_edges[4];                        /* 0.75 1.5 2.5 20 (4th unused, C17)      */
    double  speed_wet[4];                       /* 1.8 0.9 0.45 0.0 m/s                   */
    /* social force (C24-C26) */
    double  tau, A_s, B_s, radius, R_int, vmax_factor;   /* .5 25 .08 .3 1.0 1.3          */
    /* navigation (C28) */
    int32_t        n_targets;
    const uint8_t *nav_dir;                     /* [n_targets][ny*nx] direction code      */
    int32_t        exit_target, storage_target, drop_target;
    int32_t        n_exit_cells;
    const int32_t *exit_cells;                  /* [n_exit_cells], at most 16             */
    int32_t        storage_cell, drop_cell, arrive_cells;   /* arrival = Chebyshev cell distance <= arrive_cells (C29, C31) */
    /* sandbag barrier (C31-C36) */
    int32_t        n_line;
    const int32_t *line_cells;                  /* [n_line] barrier cells in filling order, not solid */
    int32_t        bags_per_cell_layer, n_layers;
    double  layer_thickness, t_pick, t_drop;    /* 0.25 m, 30 s, 30 s                     */
    double  t_end;                              /* steps are no-ops once t >= t_end; INFINITY = off */
    /* accuracy of the flood step: 0 or 1 = the paper's scheme, "reduced to first-order accuracy"
     * (P:L97); 2 = the second-order MUSCL-Hancock scheme it was reduced from (reading
     * M1-M7 of DESIGN.md): minmod slopes, Hancock half-step predictor, same HLLC flux, hydrostatic
     * reconstruction, friction and CFL rule */
    int32_t flood_order;
    /* open edges, entrance doors, pre-flood phase, evacuation trigger (P:L136, L164,
     * L180-186; readings D1-D9 of DESIGN.md).  All zero = the closed hall of the five configs. */
    int32_t        open_sides;                  /* bit (1 << SIM_SIDE_*): that domain edge is open (transmissive ghost) except at
                                                   inflow faces (D1); the flood kernel is then variant 0 (or 5 with flood_order 2) */
    int32_t        n_doors;                     /* entrance doors, at most 16 (seven, probability 1/7 each)       */
    const int32_t *door_cells;                  /* [n_doors] walkable cell of each door                                   */
    const int32_t *door_target;                 /* [n_doors] navigation field (index into nav_dir) that leads to it       */
    double         spawn_rate;                  /* pedestrians entering per second and door while not triggered  */
    int32_t        target_population;           /* doors let somebody in only while fewer pedestrians are active */
    uint64_t       spawn_seed;                  /* key of the Philox4x32-10 draws of a newcomer (D5)                      */
    double         spawn_vpref_lo, spawn_vpref_hi;   /* dry walking speed of a newcomer: uniform in [lo, hi)              */
} sim_params_t;

typedef struct {
    double  t, dt;                              /* time reached; dt of the NEXT step      */
    int64_t step;
    double  volume, max_h, max_hr;              /* volume summed in fp64                  */
    int64_t hist[6];                            /* dry low medium high highest exited     */
    int64_t neg_depth_clamps;                   /* C12                                    */
    double  clamped_volume;
    int32_t cursor, layer, bags, barrier_complete;
    int64_t deposits;
    double  outflow_volume;                     /* left through open edges (D1): V = V0 + inflow - outflow + clamped */
    int64_t spawned;                            /* newcomers so far (D3)                  */
    int32_t triggered;                          /* 1 once a wet cell exists (D7)  */
} sim_stats_t;

/* Bytes of device workspace sim_create needs for this problem. */
int sim_workspace_bytes(const sim_grid_t *grid, int32_t n_peds, const sim_params_t *params,
                        size_t *bytes);

/* Validate, place all state in device memory, upload, compute the first dt. */
int sim_create(const sim_grid_t *grid, const sim_topo_t *topo, const void *manning /* [ny*nx] real */,
               const sim_peds_t *peds, const sim_params_t *params,
               void *workspace /* device or NULL */, void *cuda_stream, sim_t **out);

/* Enqueue n coupled steps on the stream; asynchronous; dt and t stay on the device. */
int sim_step(sim_t *s, int64_t n);

/* Flood agents' recorded fields: depth, velocities (0 where h <= h_dry, C8), bed,
 * hazard rate.  Each [ny*nx] real; any pointer may be NULL. */
int sim_read_flood(sim_t *s, void *h, void *u, void *v, void *z, void *hr);
/* The conserved state [h, hu, hv] itself. */
int sim_read_conserved(sim_t *s, void *h, void *qx, void *qy);
/* N_p per cell as used by the most recent step (saturated at 255). [ny*nx] */
int sim_read_occupancy(sim_t *s, uint8_t *np_cell);
/* Pedestrians in ORIGINAL index order, length n: position, velocity (real), risk
 * state, FSM, active flag (0 = has left), containing cell, wait timer (real). Any may be NULL. */
int sim_read_peds(sim_t *s, void *x, void *y, void *vx, void *vy, uint8_t *state, uint8_t *fsm,
                  uint8_t *active, int32_t *cell, void *timer);
int sim_get_stats(sim_t *s, sim_stats_t *out);

/* ---- row slabs across GPUs (SURVEY 8f-4, S:8e) ----
 * The flood grid is cut into n <= 8 slabs of whole rows, one handle per slab, in row order, each on
 * its own device (or, for testing, several on one device); all slabs but the last have the same
 * number of rows.  sim_slab_link makes the handles one simulation:
 *   - the flood kernel of a slab reads the one halo row it needs from the neighbour slab IN PLACE
 *     (peer memory: the handles must be in one process with peer access, which this call enables;
 *     no halo buffers, no exchange kernel); "immediate neighbours";
 *   - the global time step is the minimum over the slabs: one 8-byte max-reduction of the wave
 *     speed per step;
 *   - all pedestrians live on handles[0] (the other handles are created with n = 0): its
 *     pedestrian kernels sample depth and velocity of whichever slab holds the cell, write N_p
 *     there and raise the bed there, again in place.
 * Flood kernels: variant 4 (nx a multiple of 256) or 0.  Not combined with open edges or flood_order 2.
 * sim_slab_step advances all slabs by n coupled steps (host-sequenced launches on the handles'
 * streams, events between them; no kernel waits on another); sim_step on a linked handle fails.
 * Results are bit-identical to the single-handle run of the whole grid. */
int sim_slab_link(sim_t *const *handles, int32_t n);
int sim_slab_step(sim_t *const *handles, int32_t n, int64_t steps);

/* The same slabs with ONE PROCESS PER GPU (torch.distributed; binding.SlabRank).  A slab describes
 * what it lends to the others -- device addresses in ITS address space and the base of its
 * workspace; the other processes map that workspace (CUDA IPC: torch's shared CUDA tensors), rebase
 * the addresses into their own address space and attach all n descriptions, their own included, in
 * row order.  One step of a rank is then
 *     sim_slab_enqueue(s, 0)   pedestrian step and binning chain of the next step (the rank that holds
 *                              the pedestrians), then the flood kernel of this slab
 *     all-reduce MAX over the ranks of the 8 bytes at `lam_bits` (NCCL; it is also the only barrier
 *                              the step needs: every peer access of step n is ordered before it)
 *     sim_slab_enqueue(s, 1)   tail: t += dt, next dt from the global wave speed
 * and after attaching, once: sim_slab_enqueue(s, 2) (the pedestrians binned and counted into the N_p
 * of whichever slab holds their cell, wave speed of the initial state), the same all-reduce,
 * sim_slab_enqueue(s, 3).  The same three calls, on every rank, after anything that invalidates the
 * bins (sim_write_peds, sim_set_deterministic, ...): phase 0 fails with SIM_EINVAL otherwise, because
 * bins made inside phase 0 would put N_p into another process's slab while its flood kernel reads it.  No doors in this mode (newcomers are placed by the tail, after
 * the binning chain has run).  One peer access comes AFTER the all-reduce: the tail of the first slab
 * raises the bed where responders have dropped sandbags, and nothing orders that write
 * against another process's next flood kernel.  sim_slab_attach therefore fails with SIM_EINVAL
 * unless every barrier cell lies in the first slab's rows; sim_slab_link has no such limit. */
typedef struct {
    int32_t  j0, ny;                            /* rows [j0, j0 + ny) of the grid                     */
    uint64_t h[2], qx[2], qy[2], zs, occ, ctl;  /* device addresses of the slab's arrays              */
    uint64_t lam_bits;                          /* device address of the 8-byte wave-speed word       */
    uint64_t workspace, workspace_bytes;        /* the allocation all of them live in                 */
} sim_slab_desc_t;
int sim_slab_describe(sim_t *s, sim_slab_desc_t *out);
int sim_slab_attach(sim_t *s, int32_t rank, int32_t n, const sim_slab_desc_t *descs);
int sim_slab_enqueue(sim_t *s, int32_t phase);

/* ---- the CFL time step of a flood state, for callers that must not allocate device memory ----
 * Who this is for.  Everything above needs device memory from somewhere: sim_create either calls cudaMalloc or
 * is handed a workspace the caller allocated.  Some callers can do neither at the moment they need a time step:
 *   - a host application whose own pool allocator (PyTorch's caching allocator, an RMM pool, a rendering or
 *     solver framework's arena) already owns practically all of the GPU's memory, so that a cudaMalloc from a
 *     guest library fails or evicts what the host keeps resident;
 *   - a loop with a latency budget (a live coupled run, a real-time viewer), where cudaMalloc / cudaFree are not
 *     acceptable because they may synchronise the whole device and take an unbounded time;
 *   - a plug-in that is only given pointers to the host solver's depth and discharge fields and has no
 *     permission to create device buffers of its own.
 * Such a caller holds h, qx, qy (and perhaps a solid mask) in device memory already and wants the one global
 * number the method derives from them every step: the largest wave speed over the wet cells and the time step
 * the CFL criterion allows.
 *
 *   lam = max over cells with mask == 0 and h > h_dry of max((|qx/h| + sqrt(g h)) / dx, (|qy/h| + sqrt(g h)) / dy)
 *   dt  = lam > 0 ? min(dt_max, cfl / lam) : dt_max
 *
 * computed in the precision real_bits names, cell by cell as sim_create / sim_step compute it (without their
 * clamp to t_end), the maximum taken exactly.  out[0] = lam, out[1] = dt.
 *
 * Arguments: h, qx, qy are DEVICE pointers to n_cells reals each; mask is a DEVICE pointer to n_cells bytes
 * (non-zero = solid cell, skipped) or NULL; out is a DEVICE pointer to two doubles, written by the kernel; the
 * caller owns all of them.  cuda_stream as elsewhere.  The call only enqueues work (one 8-byte memset and one
 * kernel) on the stream of the CURRENT device, which must be the device the pointers live on, and returns;
 * read `out` after synchronising that stream.  n_cells = 0 gives lam = 0, dt = dt_max.
 *
 * Scratch.  The block-wise partial maxima and a counter live in a fixed array inside the library's device image
 * (256 KiB + 256 bytes on every GPU that loads libfloodped.so, released when the process exits), not in
 * allocated memory.  Hence the limit: n_cells <= SIM_CFL_STATIC_MAX_CELLS (2^28 = a 16384 x 16384 grid); a
 * larger n_cells is refused with SIM_EINVAL and a message naming the limit.  The entry point calls no cudaMalloc,
 * cudaFree or allocating library routine.
 *   - The first call on each device looks up the array's device address (cudaGetSymbolAddress, which may load
 *     the library's device code); make that first call outside any stream capture.
 *   - There is ONE such array per device, shared by every call from every thread and stream, and it keeps what
 *     the previous call left.  Each call re-zeroes the counter it depends on, so calls that follow one another on
 *     one stream need nothing from the caller; calls that may overlap on the GPU (different streams, or different
 *     threads' streams, without an event between them) race on it and return garbage.  Serialise them.
 * Errors: SIM_EINVAL (NULL pointer, size beyond the limit, non-positive dx dy g cfl h_dry dt_max, real_bits),
 * SIM_ECUDA; the text is at sim_last_error(NULL). */
#define SIM_CFL_STATIC_MAX_CELLS (1 << 28)
int sim_cfl_dt_static(const void *h, const void *qx, const void *qy, const uint8_t *mask, int64_t n_cells,
                      int32_t real_bits, double dx, double dy, double g, double h_dry, double cfl, double dt_max,
                      void *cuda_stream, double *out /* DEVICE, [2]: lam, dt */);

/* ============================================================================================
 * Everything above is the product ABI of SURVEY 8(b).  Below: TEST AND TUNING HOOKS -- state
 * re-injection for the parity tests, kernel selection and per-kernel timing for measurement.
 * A user of the simulator needs none of them.  (SURVEY 8(b) deviations, recorded in DESIGN.md 1:
 * sim_read_peds / sim_write_peds take separate arrays incl. `active` and `timer`.)
 * ============================================================================================ */
/* The same n steps launched kernel by kernel (no graph) with a CUDA event before each launch;
 * synchronises.  kernel_ms[8] receives the summed device time in ms of: 0 bin count, 1 bin scan,
 * 2 scatter, 3 pedestrian step, 4 flood step, 5 tail, 6 occupancy (N_p per cell); 7 unused.  For measurement. */
int sim_step_profiled(sim_t *s, int64_t n, double *kernel_ms);


/* Bin the pedestrians of the current level without stepping: key[n] in original order (bin
 * index, n_bins for inactive), order[n] = original index held by each sorted slot,
 * start[n_bins+2] exclusive scan (start[n_bins+1] = n).  Bins are k x k cells,
 * k = ceil(R_int / min(dx,dy)) (C26).  Pointers may be NULL; HOST or DEVICE. */
int sim_bin_peds(sim_t *s, int32_t *key, int32_t *order, int32_t *start,
                 int32_t *n_bins_x, int32_t *n_bins_y, int32_t *k);
/* Re-inject state (HOST pointers, NULL = keep). */
int sim_write_flood(sim_t *s, const void *h, const void *qx, const void *qy, const void *z);
int sim_write_peds(sim_t *s, const void *x, const void *y, const void *vx, const void *vy,
                   const uint8_t *fsm, const uint8_t *active, const void *timer);
int sim_set_time(sim_t *s, double t, double dt);
int sim_set_barrier(sim_t *s, int32_t cursor, int32_t layer, int32_t bags, int32_t complete);
/* The device's Philox4x32-10 (D5) on n (counter[4], key[2]) rows of `in` -> n rows of 4 words in
 * `out`; HOST pointers; s only names the device and stream. */
int sim_test_philox(sim_t *s, const uint32_t *in, uint32_t *out, int32_t n);
/* Choose the flood kernel: 0 = one thread per cell, 4 faces each (any nx); 1 = 64x16 tiles, each
 * face once, shared-memory staging (nx % 4 == 0); 2 = row-marching strips of 256 columns, each
 * face once, rows prefetched in registers (any nx); 3 = as 2 with two columns per thread and
 * 64/128-bit accesses (nx % 2 == 0); 4 = as 3 with the rows of interior chunks brought in by TMA
 * bulk copies into a shared-memory ring (nx % 16 == 0).
 * Default: from 2^22 cells 4 (else 3, else 2), below that 1 (or 0).  With flood_order = 2 the
 * kernel is the MUSCL-Hancock tile kernel (reported as variant 5) and cannot be changed. */
int sim_set_flood_variant(sim_t *s, int32_t variant);
int sim_get_flood_variant(const sim_t *s);         /* the kernel in use, or SIM_EINVAL */
/* Rows per chunk of the row-marching kernels (8..64; default chosen by sim_create). Tuning hook. */
int sim_set_march_rows(sim_t *s, int32_t rows);
/* 1 (default): the pedestrian step runs as a parallel branch of the step graph beside the flood
 * step (both read level n only); 0: every kernel of the step in one chain.  Same results. */
int sim_set_overlap(sim_t *s, int32_t on);
/* 1 (default): the TMA march kernel skips chunks whose cells, and whose neighbour segments, hold exact
 * zeros (dry ground: every flux is zero, the result is zeros), reading and writing nothing for them;
 * 0: every chunk is computed.  Same results bit for bit. */
int sim_set_dry_skip(sim_t *s, int32_t on);
/* Reproducible pedestrian results (the GPU model "reproduced the same predictions as the
 * sequential counterpart"; SURVEY 8a-B "stable-enough scatter").
 * 0 (default): the slot an agent takes inside its sort bin is the order in which warps reach an
 * atomic counter; the social force is summed in slot order, so two runs of the same
 * input differ in the last bits of every agent that has neighbours, and a crowd at an exit
 * amplifies that within a few hundred steps.
 * 1: two more kernels per step order every bin by ORIGINAL agent id (O(agents per bin) per agent):
 * the forces are summed bin by bin in increasing id -- the order of the oracle's cell lists -- and
 * the results are the same bits on every run, on any number of row slabs, and in whatever order the
 * agents were written.  Inactive slots (behind the last bin) keep their arrival order.
 * Takes effect from the next step; the flood kernels are deterministic either way. */
int sim_set_deterministic(sim_t *s, int32_t on);
/* Number of kernels sim_step launches per coupled step (for launch accounting). */
int sim_kernels_per_step(const sim_t *s);

const char *sim_last_error(const sim_t *s);     /* s may be NULL: error of the last failed create */
void sim_destroy(sim_t *s);

#ifdef __cplusplus
}
#endif
#endif
