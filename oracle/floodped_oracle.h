/*
 * floodped_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded fp64 CPU statement of the coupled
 * flood-pedestrian timestep of Shirvani, Kesserwani & Richmond,
 * "Agent-based simulator of dynamic flood-people interactions"
 * (arXiv 1908.05232).  Citations "P:L<n>" are line numbers of the paper text
 * (PAPER.md); "S:8c-Cnn" are the readings listed in SURVEY.md section 8(c)
 * and repeated in DESIGN.md where the paper is silent.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or helper with the CUDA path (paper_1908_05232_b200/csrc) and
 * neither includes the other.
 *
 * Parity pins (tests/test_oracle_*.py): lake at rest / island (C-property),
 * closed-domain mass conservation, Stoker + Ritter analytical dam breaks with
 * grid refinement, transposition symmetry, exact friction closed form, CFL
 * closed form, inflow volume, paper HR values, Table 1
 * (P:L114-120), roughness rule, brute-force O(N^2) neighbour search,
 * free-walk closed form, responder FSM timeline, barrier integer arithmetic.
 * PARITY UNPINNED: the paper's count of 3484 sandbags per layer is
 * not reproducible from its own dimensions (S:8c-C32); bags_per_cell_layer is
 * an input here.
 */
#ifndef FLOODPED_ORACLE_H
#define FLOODPED_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

/* sides of a cell, used for inflow faces */
enum { ORC_W = 0, ORC_E = 1, ORC_S = 2, ORC_N = 3 };
/* flood-risk states, Table 1 plus "dry" (S:8c-C17) */
enum { ORC_DRY = 0, ORC_LOW = 1, ORC_MEDIUM = 2, ORC_HIGH = 3, ORC_HIGHEST = 4 };
/* responder finite-state machine; evacuees stay in EVACUATE */
enum { ORC_EVACUATE = 0, ORC_TO_STORAGE = 1, ORC_PICKING = 2, ORC_TO_BARRIER = 3, ORC_DROPPING = 4 };

typedef struct {
    /* grid: row-major [j][i], cell (i,j) has centre ((i+.5)dx,(j+.5)dy) */
    int nx, ny;
    double dx, dy;
    int real_bits;               /* 32: integer-valued decisions are replayed in float (see .c) */
    const double *z;             /* [ny*nx] bed elevation                                  */
    const double *manning;       /* [ny*nx] initial n_M                                    */
    const unsigned char *mask;   /* [ny*nx] 1 = solid / impassable, may be NULL            */
    const double *h0, *u0, *v0;  /* initial depth and velocities, may be NULL (= 0)        */
    /* pedestrians */
    int n_peds;
    const double *px, *py, *pvx, *pvy, *pvpref;
    const unsigned char *prole;  /* 0 evacuee, 1 responder */
    /* hydrodynamics */
    double g, cfl, dt_max, h_dry;
    int couple_roughness, n_cap;
    int n_inflow;
    const int *inflow_cell;            /* cell index j*nx+i, on the domain edge named by side */
    const unsigned char *inflow_side;  /* ORC_W/E/S/N */
    int n_hydro;
    const double *hydro_t, *hydro_q;   /* piecewise-linear Q(t), m3/s */
    /* Table 1 */
    double hr_edges[4];          /* .75 1.5 2.5 20 (the last is not used, S:8c-C17) */
    double speed_wet[4];         /* 1.8 .9 .45 0 */
    /* social force (S:8c-C24) */
    double tau, A_s, B_s, radius, R_int, vmax_factor;
    /* navigation (S:8c-C28) */
    int n_targets;
    const unsigned char *nav_dir;      /* [n_targets][ny*nx], 0..7 = E,NE,N,NW,W,SW,S,SE ; 255 none */
    int exit_target, storage_target, drop_target;
    int n_exit_cells;
    const int *exit_cells;
    int storage_cell, drop_cell, arrive_cells;
    /* sandbag barrier */
    int n_line;
    const int *line_cells;
    int bags_per_cell_layer, n_layers;
    double layer_thickness, t_pick, t_drop;
    double t_end;
    /* ---- widened scope; zero-initialised = the paper's first-order closed-wall scheme ---- */
    int flood_order;             /* 0 or 1: first order ("reduced to first-order accuracy");
                                    2: MUSCL-Hancock, the second-order scheme it was reduced from (M1-M7) */
    /* SURVEY 8f-3 (readings D1-D9 of DESIGN.md): open boundary, entrance
     * doors with spawning, pre-flood wandering, evacuation trigger */
    int open_sides;              /* bit (1 << ORC_W/E/S/N): that domain edge is open (transmissive ghost) except at inflow faces (D1) */
    int n_doors;                 /* entrance doors (7, "equal probability of 1/7"), at most 16 */
    const int *door_cells;       /* [n_doors] walkable cell of each door */
    const int *door_target;      /* [n_doors] index of the navigation field that leads to it */
    double spawn_rate;           /* pedestrians entering per second per door ("constant rate of 10 ... per entrance") (D3) */
    int target_population;       /* doors spawn only while fewer pedestrians are active ("maintain a total of 1000") */
    unsigned long long spawn_seed;     /* key of the counter-based generator (Philox4x32-10) that draws a newcomer (D5) */
    double spawn_vpref_lo, spawn_vpref_hi;   /* dry walking speed of a newcomer, uniform in [lo, hi) */
    const unsigned char *pactive0;     /* [n_peds] initial active flag per slot, NULL = all active; inactive slots are free for newcomers */
} orc_config;

/* pedestrians that entered through a door and walk to a destination door before the flood
 * (P:L164, L186): fsm = ORC_WANDER + destination door; they become evacuees at the trigger */
enum { ORC_WANDER = 8 };

typedef struct {
    double t, dt;
    long long step;
    double volume, max_h, max_hr;
    long long hist[6];           /* dry low medium high highest exited */
    long long neg_depth_clamps;
    double clamped_volume;
    int cursor, layer, bags, barrier_complete;
    long long deposits;
    double outflow_volume;       /* volume that left through open edges (D1): V = V0 + inflow - outflow + clamped */
    long long spawned;           /* newcomers so far (D3) */
    int triggered;               /* 1 once a wet cell exists: no more entries, everybody evacuates (D7) */
} orc_stats;

typedef struct orc_sim orc_sim;

/* ---- building blocks, exported so that tests can pin each one ---- */

/* Riemann flux across one face on reconstructed states, S:8c-O2 (HLLC; P:L97 cites the scheme).
 * (hL,unL,utL | hR,unR,utR) -> F[0]=mass, F[1]=normal momentum, F[2]=tangential momentum. */
void orc_riemann_flux(double g, double hL, double unL, double utL,
                      double hR, double unR, double utR, double F[3]);
/* One face between cell i (left/lower) and cell k (right/upper) with bed elevations: hydrostatic
 * reconstruction + flux; Fi[1] / Fk[1] are the normal-momentum fluxes as seen by each side. */
void orc_face(double g, double hi, double uni, double uti, double zi,
              double hk, double unk, double utk, double zk,
              double F[3], double *Fn_seen_by_i, double *Fn_seen_by_k);
/* minmod slope limiter of the second-order variant (M1) */
double orc_minmod(double a, double b);
/* pointwise semi-implicit Manning friction, S:8c-O2.4 */
void orc_friction(double g, double n, double dt, double h_dry, double h,
                  double *qx, double *qy);
/* CFL time step of one cell, S:8c-O5 */
double orc_cell_dt(double g, double cfl, double dx, double dy, double h, double u, double v);
/* HR = (max(|u|,|v|)+0.5) h; real_bits 32 evaluates in float */
double orc_hazard_rate(int real_bits, double h, double u, double v);
/* Table 1 class from h and HR (S:8c-C17) */
int orc_risk_state(int real_bits, double h, double hr, double h_dry, const double edges[4]);
/* n_eff = n0 (1 + min(Np, cap)) (S:8c-C22/C23) */
double orc_roughness(double n0, int Np, int cap);
/* piecewise-linear hydrograph */
double orc_hydrograph(int n, const double *t, const double *q, double time);
/* social acceleration on agent i by brute force over all agents (S:8c-O3.4) */
void orc_social_bruteforce(int n, const double *x, const double *y, const unsigned char *active,
                           double A_s, double B_s, double radius, double R_int,
                           int i, double *ax, double *ay);

/* Philox4x32-10 (Salmon et al. 2011): counter c[4], key k[2] -> out[4] (D5) */
void orc_philox4x32(const unsigned int c[4], const unsigned int k[2], unsigned int out[4]);

/* ---- the simulator ---- */
orc_sim *orc_create(const orc_config *cfg);
void orc_destroy(orc_sim *s);
int  orc_step(orc_sim *s, long long n);
void orc_get_stats(orc_sim *s, orc_stats *out);
/* any output pointer may be NULL */
void orc_read_flood(orc_sim *s, double *h, double *u, double *v, double *z, double *hr);
void orc_read_conserved(orc_sim *s, double *h, double *qx, double *qy);
void orc_read_occupancy(orc_sim *s, int *Np);                 /* of the most recent step */
void orc_read_peds(orc_sim *s, double *x, double *y, double *vx, double *vy,
                   unsigned char *state, unsigned char *fsm, unsigned char *active,
                   int *cell, double *timer);
/* social acceleration of every agent at the current level via the oracle's own cell list */
void orc_social_celllist(orc_sim *s, double *ax, double *ay);
/* bin key of every agent, per-bin count and exclusive start (S:8a-B); bins are k x k cells,
 * k = ceil(R_int/dx); returns number of bins, writes nbx/nby/k when non-NULL */
int  orc_binning(orc_sim *s, int *key, int *count, int *start, int *nbx, int *nby, int *k);
/* test hooks: re-inject state */
void orc_write_flood(orc_sim *s, const double *h, const double *qx, const double *qy, const double *z);
void orc_write_peds(orc_sim *s, const double *x, const double *y, const double *vx, const double *vy,
                    const unsigned char *fsm, const unsigned char *active, const double *timer);
void orc_set_time(orc_sim *s, double t, double dt);
void orc_set_barrier(orc_sim *s, int cursor, int layer, int bags, int complete);

#ifdef __cplusplus
}
#endif
#endif
