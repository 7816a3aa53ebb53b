/*
 * floodped_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see floodped_oracle.h).
 *
 * One coupled step n -> n+1 (S:8c "O1..O5"), every read at level n (the paper's
 * "simultaneous" update):
 *   O1 occupancy N_p -> roughness
 *   O2 flood cells, Eq. (2)
 *   O3 pedestrians
 *   O4 sandbag barrier -> z
 *   O5 t += dt ; CFL dt for the next step P:L174
 *
 * Everything is double.  When real_bits == 32 the handful of expressions that
 * decide an INTEGER output (cell index, risk state, timer expiry) are rounded to
 * float after every single operation through rnd(): for + - * / on float inputs,
 * double arithmetic followed by one rounding to float equals the float operation
 * (53 >= 2*24+2), so both sides take those decisions in the same precision.
 *
 * No blocking, fusion or reordering: loops over cells, faces and agents as written.
 *
 * Widened scope: flood_step_muscl (8f-2, readings M1-M7) and, for 8f-3 (P:L136, L164,
 * L180-186; readings D1-D9 of DESIGN.md), open domain edges, entrance doors that let pedestrians
 * in before the flood, their wandering to a destination door, and the evacuation trigger.
 */
#include "floodped_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

struct orc_sim {
    orc_config c;                 /* scalar copy; pointers below are owned copies */
    int ncell;
    double *z, *n0, *h, *qx, *qy, *h1, *qx1, *qy1;
    double *fv[4][4];             /* second-order variant: predicted (h, qx, qy, z) at the W, E, S, N face of every cell */
    unsigned char *mask;
    int *Np;
    int *inflow_mult[4];          /* per side, how many listed inflow faces sit on that cell side */
    double inflow_length;         /* total length of all inflow faces */
    int *inflow_cell; unsigned char *inflow_side;
    double *hydro_t, *hydro_q;
    unsigned char *nav_dir;
    int *exit_cells, *line_cells;
    /* pedestrians */
    int np;
    double *x, *y, *vx, *vy, *vpref, *timer;
    double *x1, *y1, *vx1, *vy1, *timer1;
    unsigned char *role, *state, *fsm, *active, *state1, *fsm1, *active1;
    int *cell;                    /* level-n cell of each agent in the most recent step */
    /* cell list */
    int kbin, nbx, nby;
    int *head, *next;
    /* scalars */
    double t, dt;
    long long step, deposits, neg_clamps;
    double clamped_volume;
    int cursor, layer, bags, complete;
    /* SURVEY 8f-3 */
    int *door_cells, *door_target;
    double door_credit[16];       /* fractional newcomers owed by each door (D3) */
    double outflow_volume;
    long long spawned;
    int triggered;
};

static double rnd(const orc_sim *s, double v) { return s->c.real_bits == 32 ? (double)(float)v : v; }
static double rnd_bits(int real_bits, double v) { return real_bits == 32 ? (double)(float)v : v; }

/* ------------------------------------------------------------------ building blocks */

void orc_riemann_flux(double g, double hL, double unL, double utL,
                      double hR, double unR, double utR, double F[3])
{
    /* S:8c-O2.1: both dry -> 0 */
    if (hL <= 0.0 && hR <= 0.0) { F[0] = F[1] = F[2] = 0.0; return; }
    double cL = sqrt(g * hL), cR = sqrt(g * hR);
    double sL, sR;
    if (hL <= 0.0) {                       /* dry on the left */
        sL = unR - 2.0 * cR; sR = unR + cR;
    } else if (hR <= 0.0) {                /* dry on the right */
        sL = unL - cL; sR = unL + 2.0 * cL;
    } else {                               /* two-rarefaction estimates (S:8c-C3) */
        double us = 0.5 * (unL + unR) + cL - cR;
        double cs = 0.5 * (cL + cR) + 0.25 * (unL - unR);
        sL = fmin(unL - cL, us - cs);
        sR = fmax(unR + cR, us + cs);
    }
    /* physical fluxes F = (h u, h u^2 + g h^2/2, .) */
    double FL0 = hL * unL, FL1 = hL * unL * unL + 0.5 * g * hL * hL;
    double FR0 = hR * unR, FR1 = hR * unR * unR + 0.5 * g * hR * hR;
    if (sL >= 0.0)      { F[0] = FL0; F[1] = FL1; }
    else if (sR <= 0.0) { F[0] = FR0; F[1] = FR1; }
    else {
        F[0] = (sR * FL0 - sL * FR0 + sL * sR * (hR - hL)) / (sR - sL);
        F[1] = (sR * FL1 - sL * FR1 + sL * sR * (hR * unR - hL * unL)) / (sR - sL);
    }
    /* contact wave: tangential momentum is advected by the mass flux */
    double num = sL * hR * (unR - sR) - sR * hL * (unL - sL);
    double den = hR * (unR - sR) - hL * (unL - sL);
    double sM = (den == 0.0) ? 0.0 : num / den;
    F[2] = F[0] * (sM >= 0.0 ? utL : utR);
}

void orc_face(double g, double hi, double uni, double uti, double zi,
              double hk, double unk, double utk, double zk,
              double F[3], double *Fn_i, double *Fn_k)
{
    /* hydrostatic reconstruction (S:8c-C4; the "terrain integration and wetting-and-drying
     * treatment" of P:L108): face bed = max, depths cut at the face bed, velocities kept */
    double zf = fmax(zi, zk);
    double his = fmax(0.0, (hi + zi) - zf);
    double hks = fmax(0.0, (hk + zk) - zf);
    orc_riemann_flux(g, his, uni, uti, hks, unk, utk, F);
    /* bed-slope source folded into the face: each side sees F[1] - g h*^2/2 */
    *Fn_i = F[1] - 0.5 * g * his * his;
    *Fn_k = F[1] - 0.5 * g * hks * hks;
}

void orc_friction(double g, double n, double dt, double h_dry, double h, double *qx, double *qy)
{
    if (h > h_dry) {
        double D = 1.0 + dt * g * n * n * sqrt((*qx) * (*qx) + (*qy) * (*qy)) / pow(h, 7.0 / 3.0);
        *qx /= D; *qy /= D;
    } else { *qx = 0.0; *qy = 0.0; }
}

double orc_cell_dt(double g, double cfl, double dx, double dy, double h, double u, double v)
{
    double c = sqrt(g * h);
    return cfl * fmin(dx / (fabs(u) + c), dy / (fabs(v) + c));
}

double orc_hazard_rate(int real_bits, double h, double u, double v)
{
    double V = fmax(fabs(u), fabs(v));
    return rnd_bits(real_bits, rnd_bits(real_bits, V + 0.5) * h);
}

int orc_risk_state(int real_bits, double h, double hr, double h_dry, const double e[4])
{
    if (!(h > rnd_bits(real_bits, h_dry))) return ORC_DRY;   /* S:8c-C17 */
    if (hr < rnd_bits(real_bits, e[0])) return ORC_LOW;      /* half-open [lo,hi) */
    if (hr < rnd_bits(real_bits, e[1])) return ORC_MEDIUM;
    if (hr < rnd_bits(real_bits, e[2])) return ORC_HIGH;
    return ORC_HIGHEST;
}

double orc_roughness(double n0, int Np, int cap)
{
    int m = Np < cap ? Np : cap;
    return n0 * (1.0 + (double)m);                           /* n_M + N_p n_M */
}

double orc_hydrograph(int n, const double *t, const double *q, double time)
{
    if (n <= 0) return 0.0;
    if (time <= t[0]) return q[0];
    for (int k = 0; k + 1 < n; ++k)
        if (time < t[k + 1])
            return q[k] + (q[k + 1] - q[k]) * (time - t[k]) / (t[k + 1] - t[k]);
    return q[n - 1];
}

static void pair_accel(double A_s, double B_s, double radius, double R_int,
                       double xi, double yi, double xj, double yj, double *ax, double *ay)
{
    double ddx = xi - xj, ddy = yi - yj;
    double d = sqrt(ddx * ddx + ddy * ddy);
    if (d > 0.0 && d < R_int) {                              /* S:8c-O3.4, C26 */
        double f = A_s * exp((2.0 * radius - d) / B_s);
        *ax += f * ddx / d; *ay += f * ddy / d;
    }
}

void orc_social_bruteforce(int n, const double *x, const double *y, const unsigned char *active,
                           double A_s, double B_s, double radius, double R_int,
                           int i, double *ax, double *ay)
{
    *ax = 0.0; *ay = 0.0;
    for (int j = 0; j < n; ++j)
        if (j != i && active[j]) pair_accel(A_s, B_s, radius, R_int, x[i], y[i], x[j], y[j], ax, ay);
}

/* ------------------------------------------------------------------ helpers */

static void *dup_mem(const void *p, size_t bytes)
{
    void *q = malloc(bytes ? bytes : 1);
    if (p && bytes) memcpy(q, p, bytes); else memset(q, 0, bytes ? bytes : 1);
    return q;
}

static int cell_ix(const orc_sim *s, double x)
{
    double inv = rnd(s, 1.0 / s->c.dx);
    int i = (int)floor(rnd(s, x * inv));
    if (i < 0) i = 0;
    if (i > s->c.nx - 1) i = s->c.nx - 1;
    return i;
}
static int cell_iy(const orc_sim *s, double y)
{
    double inv = rnd(s, 1.0 / s->c.dy);
    int j = (int)floor(rnd(s, y * inv));
    if (j < 0) j = 0;
    if (j > s->c.ny - 1) j = s->c.ny - 1;
    return j;
}
/* is the point outside the domain or in a solid cell? (move rejection, S:8c-O3.6) */
static int blocked(const orc_sim *s, double x, double y)
{
    double fi = floor(rnd(s, x * rnd(s, 1.0 / s->c.dx)));
    double fj = floor(rnd(s, y * rnd(s, 1.0 / s->c.dy)));
    if (fi < 0.0 || fi >= (double)s->c.nx || fj < 0.0 || fj >= (double)s->c.ny) return 1;
    return s->mask[(int)fj * s->c.nx + (int)fi] != 0;
}

static int cheb(const orc_sim *s, int ca, int cb)
{
    int ai = ca % s->c.nx, aj = ca / s->c.nx, bi = cb % s->c.nx, bj = cb / s->c.nx;
    int di = abs(ai - bi), dj = abs(aj - bj);
    return di > dj ? di : dj;
}

static void velocity_of(const orc_sim *s, double h, double qx, double qy, double *u, double *v)
{
    if (h > s->c.h_dry) { *u = qx / h; *v = qy / h; } else { *u = 0.0; *v = 0.0; }
}

static double next_dt(const orc_sim *s, const double *h, const double *qx, const double *qy)
{
    /* S:8c-O5: CFL over wet cells, capped by dt_max which is also the dry value */
    double dt = s->c.dt_max;
    for (int c = 0; c < s->ncell; ++c) {
        if (s->mask[c] || !(h[c] > s->c.h_dry)) continue;
        double u, v; velocity_of(s, h[c], qx[c], qy[c], &u, &v);
        double d = orc_cell_dt(s->c.g, s->c.cfl, s->c.dx, s->c.dy, h[c], u, v);
        if (d < dt) dt = d;
    }
    return dt;
}

static void build_cell_list(orc_sim *s)
{
    int nb = s->nbx * s->nby;
    for (int b = 0; b < nb; ++b) s->head[b] = -1;
    /* insert in reverse so that each list is in increasing agent index */
    for (int i = s->np - 1; i >= 0; --i) {
        if (!s->active[i]) continue;
        int b = (cell_iy(s, s->y[i]) / s->kbin) * s->nbx + cell_ix(s, s->x[i]) / s->kbin;
        s->next[i] = s->head[b]; s->head[b] = i;
    }
}

static void social_from_list(const orc_sim *s, int i, double *ax, double *ay)
{
    *ax = 0.0; *ay = 0.0;
    int bx = cell_ix(s, s->x[i]) / s->kbin, by = cell_iy(s, s->y[i]) / s->kbin;
    for (int jy = by - 1; jy <= by + 1; ++jy)
        for (int jx = bx - 1; jx <= bx + 1; ++jx) {
            if (jx < 0 || jy < 0 || jx >= s->nbx || jy >= s->nby) continue;
            for (int j = s->head[jy * s->nbx + jx]; j >= 0; j = s->next[j])
                if (j != i)
                    pair_accel(s->c.A_s, s->c.B_s, s->c.radius, s->c.R_int,
                               s->x[i], s->y[i], s->x[j], s->y[j], ax, ay);
        }
}

/* ------------------------------------------------------------------ trigger, doors */

/* D7 ("Once a positive water depth information is received by any navigation agent"):
 * a wet cell (h > h_dry, S:8c-C5) exists */
static int any_wet(const orc_sim *s)
{
    for (int c = 0; c < s->ncell; ++c)
        if (!s->mask[c] && s->h[c] > s->c.h_dry) return 1;
    return 0;
}

/* Philox4x32-10, the counter-based generator of Salmon, Moraes, Dror & Shaw (SC'11), written out
 * from its definition: ten rounds of  (c0,c1,c2,c3) <- (hi(M1 c2)^c1^k0, lo(M1 c2), hi(M0 c0)^c3^k1, lo(M0 c0)),
 * the key bumped by the Weyl constants after every round but the last. */
void orc_philox4x32(const unsigned int c[4], const unsigned int k[2], unsigned int out[4])
{
    unsigned int c0 = c[0], c1 = c[1], c2 = c[2], c3 = c[3], k0 = k[0], k1 = k[1];
    for (int r = 0; r < 10; ++r) {
        unsigned long long p0 = 0xD2511F53ull * c0, p1 = 0xCD9E8D57ull * c2;
        unsigned int n0 = (unsigned int)(p1 >> 32) ^ c1 ^ k0, n1 = (unsigned int)p1;
        unsigned int n2 = (unsigned int)(p0 >> 32) ^ c3 ^ k1, n3 = (unsigned int)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* D3-D5: doors let pedestrians in at a constant rate while the population is below its target
 * (P:L186), each newcomer bound for one of the doors with equal probability */
static void spawn_step(orc_sim *s, double dt)
{
    const orc_config *p = &s->c;
    int pop = 0;
    for (int i = 0; i < s->np; ++i) pop += s->active[i] ? 1 : 0;
    for (int d = 0; d < p->n_doors; ++d) {
        s->door_credit[d] = s->door_credit[d] + p->spawn_rate * dt;
        while (s->door_credit[d] >= 1.0) {
            int slot = -1;
            if (pop < p->target_population)
                for (int i = 0; i < s->np; ++i) if (!s->active[i]) { slot = i; break; }   /* lowest free slot (D4) */
            if (slot < 0) { s->door_credit[d] = 1.0; break; }          /* full: the door waits, owing one */
            unsigned int ctr[4] = { (unsigned int)(s->spawned & 0xffffffffu), (unsigned int)(s->spawned >> 32), 0u, 0u };
            unsigned int key[2] = { (unsigned int)(p->spawn_seed & 0xffffffffu), (unsigned int)(p->spawn_seed >> 32) };
            unsigned int r[4];
            orc_philox4x32(ctr, key, r);
            const int dest = (int)(((unsigned long long)r[0] * (unsigned long long)p->n_doors) >> 32);
            const double ux = (double)r[1] * (1.0 / 4294967296.0), uy = (double)r[2] * (1.0 / 4294967296.0);
            const double uv = (double)r[3] * (1.0 / 4294967296.0);
            const int ci = s->door_cells[d] % p->nx, cj = s->door_cells[d] / p->nx;
            /* inside the door cell, 10 % away from its edges */
            s->x[slot] = rnd(s, (((double)ci + 0.1) + 0.8 * ux) * p->dx);
            s->y[slot] = rnd(s, (((double)cj + 0.1) + 0.8 * uy) * p->dy);
            s->vx[slot] = 0.0; s->vy[slot] = 0.0; s->timer[slot] = 0.0;
            s->vpref[slot] = rnd(s, p->spawn_vpref_lo + (p->spawn_vpref_hi - p->spawn_vpref_lo) * uv);
            s->role[slot] = 0; s->state[slot] = ORC_DRY;
            s->fsm[slot] = (unsigned char)(ORC_WANDER + dest);
            s->active[slot] = 1;
            s->cell[slot] = s->door_cells[d];
            s->door_credit[d] -= 1.0; s->spawned += 1; pop += 1;
        }
    }
}

/* ------------------------------------------------------------------ create / destroy */

orc_sim *orc_create(const orc_config *cfg)
{
    if (!cfg || cfg->nx <= 0 || cfg->ny <= 0 || !(cfg->dx > 0) || !(cfg->dy > 0)) return NULL;
    orc_sim *s = (orc_sim *)calloc(1, sizeof *s);
    s->c = *cfg;
    int nc = s->ncell = cfg->nx * cfg->ny;
    size_t nb = (size_t)nc * sizeof(double);
    s->z = dup_mem(cfg->z, nb);
    s->n0 = dup_mem(cfg->manning, nb);
    s->mask = dup_mem(cfg->mask, (size_t)nc);
    s->h = dup_mem(cfg->h0, nb);
    s->qx = dup_mem(NULL, nb); s->qy = dup_mem(NULL, nb);
    s->h1 = dup_mem(NULL, nb); s->qx1 = dup_mem(NULL, nb); s->qy1 = dup_mem(NULL, nb);
    for (int c = 0; c < nc; ++c) {
        if (s->mask[c]) { s->h[c] = 0.0; continue; }
        s->qx[c] = s->h[c] * (cfg->u0 ? cfg->u0[c] : 0.0);   /* store conserved (S:8c-C8) */
        s->qy[c] = s->h[c] * (cfg->v0 ? cfg->v0[c] : 0.0);
    }
    if (cfg->flood_order == 2)
        for (int f = 0; f < 4; ++f) for (int k = 0; k < 4; ++k) s->fv[f][k] = dup_mem(NULL, nb);
    s->Np = dup_mem(NULL, (size_t)nc * sizeof(int));
    s->inflow_length = 0.0;
    for (int k = 0; k < 4; ++k) s->inflow_mult[k] = dup_mem(NULL, (size_t)nc * sizeof(int));
    for (int f = 0; f < cfg->n_inflow; ++f) {
        int side = cfg->inflow_side[f];
        s->inflow_mult[side][cfg->inflow_cell[f]] += 1;
        s->inflow_length += (side == ORC_W || side == ORC_E) ? cfg->dy : cfg->dx;
    }
    s->inflow_cell = dup_mem(cfg->inflow_cell, (size_t)cfg->n_inflow * sizeof(int));
    s->inflow_side = dup_mem(cfg->inflow_side, (size_t)cfg->n_inflow);
    s->hydro_t = dup_mem(cfg->hydro_t, (size_t)cfg->n_hydro * sizeof(double));
    s->hydro_q = dup_mem(cfg->hydro_q, (size_t)cfg->n_hydro * sizeof(double));
    s->nav_dir = dup_mem(cfg->nav_dir, (size_t)cfg->n_targets * (size_t)nc);
    s->exit_cells = dup_mem(cfg->exit_cells, (size_t)cfg->n_exit_cells * sizeof(int));
    s->line_cells = dup_mem(cfg->line_cells, (size_t)cfg->n_line * sizeof(int));
    s->door_cells = dup_mem(cfg->door_cells, (size_t)cfg->n_doors * sizeof(int));
    s->door_target = dup_mem(cfg->door_target, (size_t)cfg->n_doors * sizeof(int));

    int np = s->np = cfg->n_peds;
    size_t pb = (size_t)np * sizeof(double);
    s->x = dup_mem(cfg->px, pb); s->y = dup_mem(cfg->py, pb);
    s->vx = dup_mem(cfg->pvx, pb); s->vy = dup_mem(cfg->pvy, pb);
    s->vpref = dup_mem(cfg->pvpref, pb);
    s->timer = dup_mem(NULL, pb);
    s->x1 = dup_mem(NULL, pb); s->y1 = dup_mem(NULL, pb);
    s->vx1 = dup_mem(NULL, pb); s->vy1 = dup_mem(NULL, pb); s->timer1 = dup_mem(NULL, pb);
    s->role = dup_mem(cfg->prole, (size_t)np);
    s->state = dup_mem(NULL, (size_t)np); s->state1 = dup_mem(NULL, (size_t)np);
    s->fsm = dup_mem(NULL, (size_t)np); s->fsm1 = dup_mem(NULL, (size_t)np);
    s->active = dup_mem(NULL, (size_t)np); s->active1 = dup_mem(NULL, (size_t)np);
    s->cell = dup_mem(NULL, (size_t)np * sizeof(int));
    for (int i = 0; i < np; ++i) {
        s->active[i] = cfg->pactive0 ? (cfg->pactive0[i] != 0) : 1;
        s->fsm[i] = s->role[i] ? ORC_TO_STORAGE : ORC_EVACUATE;
        s->cell[i] = cell_iy(s, s->y[i]) * cfg->nx + cell_ix(s, s->x[i]);
    }
    /* default cap so that nobody crosses more than one cell per step (S:8c-C10) */
    if (!(s->c.dt_max > 0.0)) {
        double vm = 1.8;
        for (int i = 0; i < np; ++i) if (s->vpref[i] > vm) vm = s->vpref[i];
        for (int k = 0; k < 4; ++k) if (cfg->speed_wet[k] > vm) vm = cfg->speed_wet[k];
        double dmin = cfg->dx < cfg->dy ? cfg->dx : cfg->dy;
        s->c.dt_max = fmin(1.0, dmin / (cfg->vmax_factor * vm));
    }
    /* sort bins: k x k cells with k dx >= R_int so that 3x3 bins are complete (S:8c-C26) */
    {
        double dmin = cfg->dx < cfg->dy ? cfg->dx : cfg->dy;
        s->kbin = (int)ceil(cfg->R_int / dmin);
        if (s->kbin < 1) s->kbin = 1;
        s->nbx = (cfg->nx + s->kbin - 1) / s->kbin;
        s->nby = (cfg->ny + s->kbin - 1) / s->kbin;
        s->head = dup_mem(NULL, (size_t)s->nbx * s->nby * sizeof(int));
        s->next = dup_mem(NULL, (size_t)np * sizeof(int));
    }
    s->t = 0.0; s->step = 0;
    s->complete = (cfg->n_line <= 0 || cfg->n_layers <= 0) ? 1 : 0;
    s->dt = next_dt(s, s->h, s->qx, s->qy);
    if (s->t + s->dt > s->c.t_end) s->dt = fmax(0.0, s->c.t_end - s->t);
    s->triggered = any_wet(s);                                  /* D8 */
    return s;
}

void orc_destroy(orc_sim *s)
{
    if (!s) return;
    void *p[] = { s->z, s->n0, s->h, s->qx, s->qy, s->h1, s->qx1, s->qy1, s->mask, s->Np,
        s->inflow_mult[0], s->inflow_mult[1], s->inflow_mult[2], s->inflow_mult[3],
        s->inflow_cell, s->inflow_side, s->hydro_t, s->hydro_q, s->nav_dir, s->exit_cells,
        s->line_cells, s->x, s->y, s->vx, s->vy, s->vpref, s->timer, s->x1, s->y1, s->vx1, s->vy1,
        s->timer1, s->role, s->state, s->fsm, s->active, s->state1, s->fsm1, s->active1, s->cell,
        s->head, s->next, s->door_cells, s->door_target };
    for (size_t k = 0; k < sizeof p / sizeof p[0]; ++k) free(p[k]);
    for (int f = 0; f < 4; ++f) for (int k = 0; k < 4; ++k) free(s->fv[f][k]);
    free(s);
}

/* ------------------------------------------------------------------ one coupled step */

/* state of the neighbour across one face of cell c: the cell itself if it is an interior
 * walkable cell, else the wall ghost (S:8c-O2.1): same h and z, normal velocity
 * negated, tangential kept */
/* D1: is the face of cell c = (i, j) towards (di, dj) an OPEN domain-edge face?  The side must be
 * flagged open and the face must not be an inflow face (those stay walls for momentum, C14). */
static int open_face(const orc_sim *s, int c, int i, int j, int di, int dj)
{
    int side;
    if (di < 0 && i == 0) side = ORC_W;
    else if (di > 0 && i == s->c.nx - 1) side = ORC_E;
    else if (dj < 0 && j == 0) side = ORC_S;
    else if (dj > 0 && j == s->c.ny - 1) side = ORC_N;
    else return 0;
    return ((s->c.open_sides >> side) & 1) && s->inflow_mult[side][c] == 0;
}

static void neighbour(const orc_sim *s, int c, int i, int j, int di, int dj,
                      double hc, double unc, double utc, double zc,
                      double *hk, double *unk, double *utk, double *zk)
{
    int ii = i + di, jj = j + dj;
    int wall = (ii < 0 || jj < 0 || ii >= s->c.nx || jj >= s->c.ny);
    /* D1: an open domain edge has a transmissive ghost (zero gradient: the cell's own state) */
    if (wall && open_face(s, c, i, j, di, dj)) { *hk = hc; *unk = unc; *utk = utc; *zk = zc; return; }
    int k = wall ? c : jj * s->c.nx + ii;
    if (!wall && s->mask[k]) wall = 1;
    if (wall) { *hk = hc; *unk = -unc; *utk = utc; *zk = zc; return; }
    double u, v; velocity_of(s, s->h[k], s->qx[k], s->qy[k], &u, &v);
    *hk = s->h[k]; *zk = s->z[k];
    if (di != 0) { *unk = u; *utk = v; } else { *unk = v; *utk = u; }
}

static void flood_step(orc_sim *s, double q_in)
{
    const double g = s->c.g, dt = s->dt, dx = s->c.dx, dy = s->c.dy;
    const int nx = s->c.nx, ny = s->c.ny;
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            int c = j * nx + i;
            if (s->mask[c]) { s->h1[c] = s->qx1[c] = s->qy1[c] = 0.0; continue; }   /* S:8c-C16 */
            double h = s->h[c], z = s->z[c], u, v;
            velocity_of(s, h, s->qx[c], s->qy[c], &u, &v);
            double hk, unk, utk, zk, F[3], Fi, Fk;

            /* EAST: cell is the left state; normal u, tangential v */
            neighbour(s, c, i, j, +1, 0, h, u, v, z, &hk, &unk, &utk, &zk);
            orc_face(g, h, u, v, z, hk, unk, utk, zk, F, &Fi, &Fk);
            double FE0 = F[0], FE1 = Fi, FE2 = F[2];
            /* WEST: cell is the right state */
            neighbour(s, c, i, j, -1, 0, h, u, v, z, &hk, &unk, &utk, &zk);
            orc_face(g, hk, unk, utk, zk, h, u, v, z, F, &Fk, &Fi);
            double FW0 = F[0], FW1 = Fi, FW2 = F[2];
            /* NORTH: cell is the lower state; normal v, tangential u */
            neighbour(s, c, i, j, 0, +1, h, v, u, z, &hk, &unk, &utk, &zk);
            orc_face(g, h, v, u, z, hk, unk, utk, zk, F, &Fi, &Fk);
            double GN0 = F[0], GN2 = Fi, GN1 = F[2];
            /* SOUTH: cell is the upper state */
            neighbour(s, c, i, j, 0, -1, h, v, u, z, &hk, &unk, &utk, &zk);
            orc_face(g, hk, unk, utk, zk, h, v, u, z, F, &Fk, &Fi);
            double GS0 = F[0], GS2 = Fi, GS1 = F[2];

            /* inflow faces: wall for momentum, prescribed mass flux into the domain
             * (S:8c-O2.1, C14) */
            FW0 += q_in * s->inflow_mult[ORC_W][c];
            FE0 -= q_in * s->inflow_mult[ORC_E][c];
            GS0 += q_in * s->inflow_mult[ORC_S][c];
            GN0 -= q_in * s->inflow_mult[ORC_N][c];

            /* volume leaving through open edge faces (D1) */
            if (open_face(s, c, i, j, +1, 0)) s->outflow_volume += dt * FE0 * dy;
            if (open_face(s, c, i, j, -1, 0)) s->outflow_volume -= dt * FW0 * dy;
            if (open_face(s, c, i, j, 0, +1)) s->outflow_volume += dt * GN0 * dx;
            if (open_face(s, c, i, j, 0, -1)) s->outflow_volume -= dt * GS0 * dx;

            /* Eq. (2) */
            double hn  = h        - dt / dx * (FE0 - FW0) - dt / dy * (GN0 - GS0);
            double qxn = s->qx[c] - dt / dx * (FE1 - FW1) - dt / dy * (GN1 - GS1);
            double qyn = s->qy[c] - dt / dx * (FE2 - FW2) - dt / dy * (GN2 - GS2);
            /* accounted clamp (S:8c-C12) */
            if (hn < 0.0) { s->clamped_volume += -hn * dx * dy; s->neg_clamps += 1; hn = 0.0; }
            /* Manning friction with the occupancy-dependent roughness */
            double n = s->c.couple_roughness ? orc_roughness(s->n0[c], s->Np[c], s->c.n_cap) : s->n0[c];
            orc_friction(g, n, dt, s->c.h_dry, hn, &qxn, &qyn);
            s->h1[c] = hn; s->qx1[c] = qxn; s->qy1[c] = qyn;
        }
}

/* ------------------------------------------------------------------ second order
 * MUSCL-Hancock variant of the flood step: the second-order scheme the paper "reduced to
 * first-order accuracy".  The paper prints none of it; this is the reading of
 * DESIGN.md M1-M7, on top of the same face flux (orc_face), clamp and friction as flood_step():
 *  M1 limited slopes of (eta, h, qx, qy), minmod, per direction; zero in a direction where the
 *     cell or a neighbour is not wet (h <= h_dry) or a neighbour is a wall (edge, solid cell):
 *     the scheme falls back to first order at wet/dry fronts and walls;
 *  M2 face values W_i +- sigma/2; bed at a face z_f = eta_f - h_f;
 *  M3 Hancock predictor: the four face values advance half a step with the physical fluxes of
 *     the cell's own face values, pressure and bed slope together as g hbar (eta_E - eta_W)
 *     (still water: no change), depth clamped at 0;
 *  M4 one Riemann flux per face on the hydrostatically reconstructed predicted face states; the
 *     momentum flux seen by a cell is F1 - g h*^2/2 + g h_f^2/2 with h_f its own face depth;
 *  M5 centred bed-slope source g (h_W + h_E)(z_W - z_E) / 2 dx of the cell's own face values;
 *  M6 update, inflow, clamp, friction as in the first-order step;  M7 same CFL rule.
 * A cell whose slopes all vanish takes exactly the first-order step. */
double orc_minmod(double a, double b)
{
    if (a * b <= 0.0) return 0.0;
    return fabs(a) < fabs(b) ? a : b;
}

enum { FV_H = 0, FV_QX = 1, FV_QY = 2, FV_Z = 3 };

static int is_wall(const orc_sim *s, int i, int j)
{
    if (i < 0 || j < 0 || i >= s->c.nx || j >= s->c.ny) return 1;
    return s->mask[j * s->c.nx + i] != 0;
}

/* M1: limited slopes of (eta, h, qx, qy) of cell c along (di, dj) */
static void muscl_slopes(const orc_sim *s, int i, int j, int di, int dj, double sl[4])
{
    sl[0] = sl[1] = sl[2] = sl[3] = 0.0;
    if (is_wall(s, i - di, j - dj) || is_wall(s, i + di, j + dj)) return;
    const int nx = s->c.nx, c = j * nx + i, a = (j - dj) * nx + (i - di), b = (j + dj) * nx + (i + di);
    if (!(s->h[c] > s->c.h_dry && s->h[a] > s->c.h_dry && s->h[b] > s->c.h_dry)) return;
    sl[0] = orc_minmod((s->h[c] + s->z[c]) - (s->h[a] + s->z[a]), (s->h[b] + s->z[b]) - (s->h[c] + s->z[c]));
    sl[1] = orc_minmod(s->h[c] - s->h[a], s->h[b] - s->h[c]);
    sl[2] = orc_minmod(s->qx[c] - s->qx[a], s->qx[b] - s->qx[c]);
    sl[3] = orc_minmod(s->qy[c] - s->qy[a], s->qy[b] - s->qy[c]);
}

/* velocity of a face value of a WET cell: q / max(h, h_dry) (continuous in h); a cell that is not
 * wet has u = v = 0 as in the first-order step */
static double face_vel(const orc_sim *s, int cell_wet, double q, double h)
{
    return cell_wet ? q / fmax(h, s->c.h_dry) : 0.0;
}

static void muscl_predict(orc_sim *s)
{
    const double g = s->c.g, dt = s->dt, dx = s->c.dx, dy = s->c.dy;
    const int nx = s->c.nx, ny = s->c.ny;
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            const int c = j * nx + i;
            if (s->mask[c]) continue;
            const double h = s->h[c], z = s->z[c], eta = h + z, qx = s->qx[c], qy = s->qy[c];
            const int wet = h > s->c.h_dry;
            double sx[4], sy[4];
            muscl_slopes(s, i, j, 1, 0, sx);
            muscl_slopes(s, i, j, 0, 1, sy);
            /* M2: face values; index 0 W, 1 E, 2 S, 3 N */
            double fe[4], fh[4], fqx[4], fqy[4], fz[4];
            for (int f = 0; f < 4; ++f) {
                const double *sl = f < 2 ? sx : sy;
                const double sg = (f == ORC_E || f == ORC_N) ? 0.5 : -0.5;
                fe[f] = eta + sg * sl[0]; fh[f] = h + sg * sl[1];
                fqx[f] = qx + sg * sl[2]; fqy[f] = qy + sg * sl[3];
                fz[f] = fe[f] - fh[f];
            }
            /* M3: Hancock predictor from the cell's own face values */
            const double uE = face_vel(s, wet, fqx[ORC_E], fh[ORC_E]), uW = face_vel(s, wet, fqx[ORC_W], fh[ORC_W]);
            const double vN = face_vel(s, wet, fqy[ORC_N], fh[ORC_N]), vS = face_vel(s, wet, fqy[ORC_S], fh[ORC_S]);
            const double dh = -0.5 * dt / dx * (fqx[ORC_E] - fqx[ORC_W]) - 0.5 * dt / dy * (fqy[ORC_N] - fqy[ORC_S]);
            const double dqx = -0.5 * dt / dx * ((fqx[ORC_E] * uE - fqx[ORC_W] * uW)
                                                + g * 0.5 * (fh[ORC_E] + fh[ORC_W]) * (fe[ORC_E] - fe[ORC_W]))
                               - 0.5 * dt / dy * (fqx[ORC_N] * vN - fqx[ORC_S] * vS);
            const double dqy = -0.5 * dt / dx * (fqy[ORC_E] * uE - fqy[ORC_W] * uW)
                               - 0.5 * dt / dy * ((fqy[ORC_N] * vN - fqy[ORC_S] * vS)
                                                  + g * 0.5 * (fh[ORC_N] + fh[ORC_S]) * (fe[ORC_N] - fe[ORC_S]));
            for (int f = 0; f < 4; ++f) {
                s->fv[f][FV_H][c] = fmax(0.0, fh[f] + dh);
                s->fv[f][FV_QX][c] = fqx[f] + dqx;
                s->fv[f][FV_QY][c] = fqy[f] + dqy;
                s->fv[f][FV_Z][c] = fz[f];
            }
        }
}

/* predicted state of cell c at its face f as (h, normal velocity, tangential velocity, z) */
static void muscl_face_state(const orc_sim *s, int c, int f, double *h, double *un, double *ut, double *z)
{
    const int wet = s->h[c] > s->c.h_dry;
    *h = s->fv[f][FV_H][c]; *z = s->fv[f][FV_Z][c];
    const double u = face_vel(s, wet, s->fv[f][FV_QX][c], *h), v = face_vel(s, wet, s->fv[f][FV_QY][c], *h);
    if (f < 2) { *un = u; *ut = v; } else { *un = v; *ut = u; }
}

static void flood_step_muscl(orc_sim *s, double q_in)
{
    const double g = s->c.g, dt = s->dt, dx = s->c.dx, dy = s->c.dy;
    const int nx = s->c.nx, ny = s->c.ny;
    muscl_predict(s);
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            const int c = j * nx + i;
            if (s->mask[c]) { s->h1[c] = s->qx1[c] = s->qy1[c] = 0.0; continue; }
            /* M4: the four faces; f = side of THIS cell, the neighbour contributes its opposite face */
            double F0[4], Fn[4], Ft[4], hf[4], zf[4];
            for (int f = 0; f < 4; ++f) {
                const int di = (f == ORC_E) - (f == ORC_W), dj = (f == ORC_N) - (f == ORC_S);
                double hi, uni, uti, zi, hk, unk, utk, zk, F[3], Fi, Fk;
                muscl_face_state(s, c, f, &hi, &uni, &uti, &zi);
                if (open_face(s, c, i, j, di, dj)) { hk = hi; unk = uni; utk = uti; zk = zi; }  /* transmissive ghost (D1) */
                else if (is_wall(s, i + di, j + dj)) { hk = hi; unk = -uni; utk = uti; zk = zi; }   /* wall ghost (S:8c-O2.1) */
                else muscl_face_state(s, (j + dj) * nx + (i + di), f ^ 1, &hk, &unk, &utk, &zk);
                if (f == ORC_E || f == ORC_N) { orc_face(g, hi, uni, uti, zi, hk, unk, utk, zk, F, &Fi, &Fk); }
                else                          { orc_face(g, hk, unk, utk, zk, hi, uni, uti, zi, F, &Fk, &Fi); }
                F0[f] = F[0]; Fn[f] = Fi + 0.5 * g * hi * hi; Ft[f] = F[2];
                hf[f] = hi; zf[f] = zi;
            }
            /* inflow faces as in the first-order step (S:8c-O2.1, C14) */
            F0[ORC_W] += q_in * s->inflow_mult[ORC_W][c];
            F0[ORC_E] -= q_in * s->inflow_mult[ORC_E][c];
            F0[ORC_S] += q_in * s->inflow_mult[ORC_S][c];
            F0[ORC_N] -= q_in * s->inflow_mult[ORC_N][c];
            if (open_face(s, c, i, j, +1, 0)) s->outflow_volume += dt * F0[ORC_E] * dy;
            if (open_face(s, c, i, j, -1, 0)) s->outflow_volume -= dt * F0[ORC_W] * dy;
            if (open_face(s, c, i, j, 0, +1)) s->outflow_volume += dt * F0[ORC_N] * dx;
            if (open_face(s, c, i, j, 0, -1)) s->outflow_volume -= dt * F0[ORC_S] * dx;
            /* M5: centred bed-slope source of the cell's own (predicted) face values */
            const double Sx = 0.5 * g * (hf[ORC_W] + hf[ORC_E]) * (zf[ORC_W] - zf[ORC_E]) / dx;
            const double Sy = 0.5 * g * (hf[ORC_S] + hf[ORC_N]) * (zf[ORC_S] - zf[ORC_N]) / dy;
            /* M6: Eq. (2) with the second-order fluxes */
            double hn  = s->h[c]  - dt / dx * (F0[ORC_E] - F0[ORC_W]) - dt / dy * (F0[ORC_N] - F0[ORC_S]);
            double qxn = s->qx[c] - dt / dx * (Fn[ORC_E] - Fn[ORC_W]) - dt / dy * (Ft[ORC_N] - Ft[ORC_S]) + dt * Sx;
            double qyn = s->qy[c] - dt / dx * (Ft[ORC_E] - Ft[ORC_W]) - dt / dy * (Fn[ORC_N] - Fn[ORC_S]) + dt * Sy;
            if (hn < 0.0) { s->clamped_volume += -hn * dx * dy; s->neg_clamps += 1; hn = 0.0; }
            double n = s->c.couple_roughness ? orc_roughness(s->n0[c], s->Np[c], s->c.n_cap) : s->n0[c];
            orc_friction(g, n, dt, s->c.h_dry, hn, &qxn, &qyn);
            s->h1[c] = hn; s->qx1[c] = qxn; s->qy1[c] = qyn;
        }
}

static void dir_vector(int code, double *ex, double *ey)
{
    static const double r = 0.70710678118654752440;
    switch (code) {
    case 0: *ex = 1;  *ey = 0;  break;   case 1: *ex = r;  *ey = r;  break;
    case 2: *ex = 0;  *ey = 1;  break;   case 3: *ex = -r; *ey = r;  break;
    case 4: *ex = -1; *ey = 0;  break;   case 5: *ex = -r; *ey = -r; break;
    case 6: *ex = 0;  *ey = -1; break;   case 7: *ex = r;  *ey = -r; break;
    default: *ex = 0; *ey = 0;
    }
}

/* returns number of deposit events D */
static long long ped_step(orc_sim *s)
{
    const orc_config *p = &s->c;
    const double dt = s->dt;
    const int complete0 = s->complete;           /* value at the start of the step (S:8c-O3.7) */
    const int triggered0 = s->triggered;         /* likewise (D7) */
    long long D = 0;
    build_cell_list(s);
    for (int i = 0; i < s->np; ++i) {
        s->x1[i] = s->x[i]; s->y1[i] = s->y[i]; s->vx1[i] = s->vx[i]; s->vy1[i] = s->vy[i];
        s->timer1[i] = s->timer[i]; s->state1[i] = s->state[i]; s->fsm1[i] = s->fsm[i];
        s->active1[i] = s->active[i];
        if (!s->active[i]) continue;
        /* 1. containing cell, sample U^n there (S:8c-C19, C20) */
        int c = s->cell[i];
        int fsm = s->fsm[i];
        /* D7: once water is in the domain, those still wandering become evacuees */
        if (fsm >= ORC_WANDER && triggered0) { fsm = ORC_EVACUATE; s->fsm1[i] = ORC_EVACUATE; }
        /* D6: a wanderer leaves through its destination door */
        if (fsm >= ORC_WANDER) {
            if (cheb(s, c, s->door_cells[fsm - ORC_WANDER]) <= p->arrive_cells) { s->active1[i] = 0; continue; }
        } else
        /* 8. exit (S:8c-C29): evaluated on the level-n cell */
        if (s->role[i] == 0 || fsm == ORC_EVACUATE) {
            int out = 0;
            for (int e = 0; e < p->n_exit_cells; ++e)
                if (cheb(s, c, s->exit_cells[e]) <= p->arrive_cells) out = 1;
            if (out) { s->active1[i] = 0; continue; }
        }
        double h = s->h[c], u, v;
        if (h > rnd(s, p->h_dry)) { u = rnd(s, s->qx[c] / h); v = rnd(s, s->qy[c] / h); }
        else { u = 0.0; v = 0.0; }
        double hr = orc_hazard_rate(p->real_bits, h, u, v);
        int st = orc_risk_state(p->real_bits, h, hr, p->h_dry, p->hr_edges);  /* Table 1 */
        s->state1[i] = (unsigned char)st;
        /* 2. desired speed (S:8c-C18) */
        double v0 = (st == ORC_DRY) ? s->vpref[i] : p->speed_wet[st - 1];
        if (fsm == ORC_PICKING || fsm == ORC_DROPPING) v0 = 0.0;              /* waiting */
        /* 3. target field by role / FSM */
        int target = p->exit_target;
        if (fsm == ORC_TO_STORAGE) target = p->storage_target;
        else if (fsm == ORC_TO_BARRIER) target = p->drop_target;
        else if (fsm >= ORC_WANDER) target = s->door_target[fsm - ORC_WANDER];
        double ex, ey;
        dir_vector(s->nav_dir[(size_t)target * s->ncell + c], &ex, &ey);
        /* 4. social repulsion from agents in adjacent bins (S:8c-C24, C26) */
        double ax, ay;
        social_from_list(s, i, &ax, &ay);
        /* 5. velocity: backward Euler on the relaxation term (S:8c-C25) */
        double wx = (s->vx[i] + dt * (v0 * ex / p->tau + ax)) / (1.0 + dt / p->tau);
        double wy = (s->vy[i] + dt * (v0 * ey / p->tau + ay)) / (1.0 + dt / p->tau);
        double wmax = p->vmax_factor * v0, wn = sqrt(wx * wx + wy * wy);
        if (wn > wmax) { double f = (wn > 0.0) ? wmax / wn : 0.0; wx *= f; wy *= f; }
        /* 6. position with axis-separated rejection at walls and solids (S:8c-C27) */
        double xn = s->x[i] + dt * wx, yn = s->y[i];
        if (blocked(s, xn, yn)) { xn = s->x[i]; wx = 0.0; }
        yn = s->y[i] + dt * wy;
        if (blocked(s, xn, yn)) { yn = s->y[i]; wy = 0.0; }
        s->x1[i] = xn; s->y1[i] = yn; s->vx1[i] = wx; s->vy1[i] = wy;
        /* 7. responder FSM on the level-n cell, once per step (S:8c-C31) */
        if (s->role[i] == 1) {
            if (fsm == ORC_TO_STORAGE) {
                if (cheb(s, c, p->storage_cell) <= p->arrive_cells) { s->fsm1[i] = ORC_PICKING; s->timer1[i] = rnd(s, p->t_pick); }
            } else if (fsm == ORC_PICKING) {
                s->timer1[i] = rnd(s, s->timer[i] - rnd(s, dt));
                if (s->timer1[i] <= 0.0) s->fsm1[i] = ORC_TO_BARRIER;
            } else if (fsm == ORC_TO_BARRIER) {
                if (cheb(s, c, p->drop_cell) <= p->arrive_cells) { s->fsm1[i] = ORC_DROPPING; s->timer1[i] = rnd(s, p->t_drop); }
            } else if (fsm == ORC_DROPPING) {
                s->timer1[i] = rnd(s, s->timer[i] - rnd(s, dt));
                if (s->timer1[i] <= 0.0) { D += 1; s->fsm1[i] = complete0 ? ORC_EVACUATE : ORC_TO_STORAGE; }
            }
        }
    }
    return D;
}

static void barrier_step(orc_sim *s, long long D)
{
    /* gather bags until one layer covers the cell, raise z by one bag thickness,
     * move to the next cell of the line, repeat N_L layers (S:8c-O4, C33, C34) */
    s->deposits += D;
    for (long long d = 0; d < D; ++d) {
        if (s->complete) break;
        s->bags += 1;
        if (s->bags == s->c.bags_per_cell_layer) {
            s->z[s->line_cells[s->cursor]] += s->c.layer_thickness;
            s->bags = 0; s->cursor += 1;
            if (s->cursor == s->c.n_line) { s->layer += 1; s->cursor = 0; }
            if (s->layer == s->c.n_layers) s->complete = 1;
        }
    }
}

int orc_step(orc_sim *s, long long n)
{
    for (long long k = 0; k < n; ++k) {
        if (s->t >= s->c.t_end) break;                      /* no-op once t_end is reached */
        /* O1 */
        memset(s->Np, 0, (size_t)s->ncell * sizeof(int));
        for (int i = 0; i < s->np; ++i) {
            if (!s->active[i]) continue;
            s->cell[i] = cell_iy(s, s->y[i]) * s->c.nx + cell_ix(s, s->x[i]);
            s->Np[s->cell[i]] += 1;                         /* all active pedestrians (S:8c-C21) */
        }
        /* O2 */
        double Q = orc_hydrograph(s->c.n_hydro, s->hydro_t, s->hydro_q, s->t);
        double q_in = (s->inflow_length > 0.0) ? Q / s->inflow_length : 0.0;
        if (s->c.flood_order == 2) flood_step_muscl(s, q_in); else flood_step(s, q_in);
        /* O3 (reads level-n flood and pedestrians) */
        long long D = ped_step(s);
        /* O4 */
        barrier_step(s, D);
        /* commit level n+1 */
        double *tp;
#define SWAP(a, b) do { tp = a; a = b; b = tp; } while (0)
        SWAP(s->h, s->h1); SWAP(s->qx, s->qx1); SWAP(s->qy, s->qy1);
        SWAP(s->x, s->x1); SWAP(s->y, s->y1); SWAP(s->vx, s->vx1); SWAP(s->vy, s->vy1);
        SWAP(s->timer, s->timer1);
#undef SWAP
        unsigned char *tb;
        tb = s->state; s->state = s->state1; s->state1 = tb;
        tb = s->fsm; s->fsm = s->fsm1; s->fsm1 = tb;
        tb = s->active; s->active = s->active1; s->active1 = tb;
        /* O5 */
        const double dt_taken = s->dt;
        s->t += s->dt;
        s->step += 1;
        /* D7: trigger on U^{n+1}; D3: doors let newcomers in (they exist from level n+1 on) */
        if (!s->triggered && any_wet(s)) s->triggered = 1;
        if (!s->triggered && s->c.n_doors > 0) spawn_step(s, dt_taken);
        s->dt = next_dt(s, s->h, s->qx, s->qy);
        if (s->t + s->dt > s->c.t_end) s->dt = fmax(0.0, s->c.t_end - s->t);
    }
    return 0;
}

/* ------------------------------------------------------------------ read / write */

void orc_get_stats(orc_sim *s, orc_stats *o)
{
    memset(o, 0, sizeof *o);
    o->t = s->t; o->dt = s->dt; o->step = s->step;
    double comp = 0.0;                       /* compensated (Neumaier) sum of the volume */
    for (int c = 0; c < s->ncell; ++c) {
        if (s->mask[c]) continue;
        double u, v; velocity_of(s, s->h[c], s->qx[c], s->qy[c], &u, &v);
        double hr = (s->h[c] > s->c.h_dry) ? orc_hazard_rate(64, s->h[c], u, v) : 0.0;
        double term = s->h[c] * s->c.dx * s->c.dy, tsum = o->volume + term;
        comp += (fabs(o->volume) >= fabs(term)) ? (o->volume - tsum) + term : (term - tsum) + o->volume;
        o->volume = tsum;
        if (s->h[c] > o->max_h) o->max_h = s->h[c];
        if (hr > o->max_hr) o->max_hr = hr;
    }
    o->volume += comp;
    for (int i = 0; i < s->np; ++i) o->hist[s->active[i] ? s->state[i] : 5] += 1;
    o->neg_depth_clamps = s->neg_clamps; o->clamped_volume = s->clamped_volume;
    o->cursor = s->cursor; o->layer = s->layer; o->bags = s->bags;
    o->barrier_complete = s->complete; o->deposits = s->deposits;
    o->outflow_volume = s->outflow_volume; o->spawned = s->spawned; o->triggered = s->triggered;
}

void orc_read_flood(orc_sim *s, double *h, double *u, double *v, double *z, double *hr)
{
    for (int c = 0; c < s->ncell; ++c) {
        double uu, vv; velocity_of(s, s->h[c], s->qx[c], s->qy[c], &uu, &vv);
        if (h) h[c] = s->h[c];
        if (u) u[c] = uu;
        if (v) v[c] = vv;
        if (z) z[c] = s->z[c];
        if (hr) hr[c] = (s->h[c] > s->c.h_dry) ? orc_hazard_rate(64, s->h[c], uu, vv) : 0.0;
    }
}

void orc_read_conserved(orc_sim *s, double *h, double *qx, double *qy)
{
    size_t nb = (size_t)s->ncell * sizeof(double);
    if (h) memcpy(h, s->h, nb);
    if (qx) memcpy(qx, s->qx, nb);
    if (qy) memcpy(qy, s->qy, nb);
}

void orc_read_occupancy(orc_sim *s, int *Np) { memcpy(Np, s->Np, (size_t)s->ncell * sizeof(int)); }

void orc_read_peds(orc_sim *s, double *x, double *y, double *vx, double *vy,
                   unsigned char *state, unsigned char *fsm, unsigned char *active,
                   int *cell, double *timer)
{
    for (int i = 0; i < s->np; ++i) {
        if (x) x[i] = s->x[i];
        if (y) y[i] = s->y[i];
        if (vx) vx[i] = s->vx[i];
        if (vy) vy[i] = s->vy[i];
        if (state) state[i] = s->state[i];
        if (fsm) fsm[i] = s->fsm[i];
        if (active) active[i] = s->active[i];
        if (cell) cell[i] = cell_iy(s, s->y[i]) * s->c.nx + cell_ix(s, s->x[i]);
        if (timer) timer[i] = s->timer[i];
    }
}

void orc_social_celllist(orc_sim *s, double *ax, double *ay)
{
    build_cell_list(s);
    for (int i = 0; i < s->np; ++i) {
        ax[i] = ay[i] = 0.0;
        if (s->active[i]) social_from_list(s, i, &ax[i], &ay[i]);
    }
}

int orc_binning(orc_sim *s, int *key, int *count, int *start, int *nbx, int *nby, int *k)
{
    int nb = s->nbx * s->nby;
    if (nbx) *nbx = s->nbx;
    if (nby) *nby = s->nby;
    if (k) *k = s->kbin;
    if (count) memset(count, 0, (size_t)nb * sizeof(int));
    for (int i = 0; i < s->np; ++i) {
        int b = nb;                                           /* inactive agents sort last */
        if (s->active[i])
            b = (cell_iy(s, s->y[i]) / s->kbin) * s->nbx + cell_ix(s, s->x[i]) / s->kbin;
        if (key) key[i] = b;
        if (count && b < nb) count[b] += 1;
    }
    if (start && count) {
        int acc = 0;
        for (int b = 0; b < nb; ++b) { start[b] = acc; acc += count[b]; }
        start[nb] = acc;
    }
    return nb;
}

void orc_write_flood(orc_sim *s, const double *h, const double *qx, const double *qy, const double *z)
{
    size_t nb = (size_t)s->ncell * sizeof(double);
    if (h) memcpy(s->h, h, nb);
    if (qx) memcpy(s->qx, qx, nb);
    if (qy) memcpy(s->qy, qy, nb);
    if (z) memcpy(s->z, z, nb);
    if (!s->triggered && any_wet(s)) s->triggered = 1;       /* D8 */
}

void orc_write_peds(orc_sim *s, const double *x, const double *y, const double *vx, const double *vy,
                    const unsigned char *fsm, const unsigned char *active, const double *timer)
{
    size_t pb = (size_t)s->np * sizeof(double);
    if (x) memcpy(s->x, x, pb);
    if (y) memcpy(s->y, y, pb);
    if (vx) memcpy(s->vx, vx, pb);
    if (vy) memcpy(s->vy, vy, pb);
    if (fsm) memcpy(s->fsm, fsm, (size_t)s->np);
    if (active) memcpy(s->active, active, (size_t)s->np);
    if (timer) memcpy(s->timer, timer, pb);
    for (int i = 0; i < s->np; ++i)
        s->cell[i] = cell_iy(s, s->y[i]) * s->c.nx + cell_ix(s, s->x[i]);
}

void orc_set_time(orc_sim *s, double t, double dt) { s->t = t; s->dt = dt; }

void orc_set_barrier(orc_sim *s, int cursor, int layer, int bags, int complete)
{
    s->cursor = cursor; s->layer = layer; s->bags = bags; s->complete = complete;
}
