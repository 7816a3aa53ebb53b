// flood_march.cuh -- variant 2 of step (F)+(T): the same flood-cell update as flood.cuh
// (Eq. (2); fluxes and sources as in DESIGN.md C2-C6, C12-C16), laid out as a
// row-marching ("2.5-D") stencil for large grids.
//
//   A CTA owns a strip of MW = 256 columns (one column per thread) and marches over R rows.
//   Per row each thread evaluates ONE x-face (its west face) and ONE y-face (its south face);
//   the south face of row j+1 is the north face of row j, so y-fluxes never leave registers.
//   The west neighbour's primitives and the east face's flux travel through a double-buffered
//   shared-memory row (one __syncthreads per row).  Rows are prefetched two iterations ahead
//   into registers with fully coalesced 128-byte warp loads, so DRAM latency overlaps the
//   arithmetic of the rows in flight; nothing is re-read except 2 halo rows per R.
//   Strip-edge faces (east) and strip-edge states (west) of all R rows are prepared once per
//   chunk by a short pre-pass.
//
//   Two instantiations: GEN = false for chunks that neither touch the domain edge nor contain or
//   touch a solid cell (no wall-ghost selects, no bounds checks, no inflow terms); GEN = true
//   otherwise.  Which one a chunk takes is precomputed per chunk (flood_chunk_flags_kernel)
//   whenever the bed is (re)loaded.
//
//   Faces whose two reconstructed depths are zero across the whole warp are skipped by a vote.
#pragma once

#include "flood.cuh"

namespace fp {

constexpr int MW = 256;               // columns per strip = threads per CTA
constexpr int MARCH_MAX_R = 64;       // rows per chunk (runtime R <= this)

template <typename T>
struct MarchSmem {
    T st[2][4][MW];                   // eta, u, v, z of the row being entered, by row parity
    T fx[2][3][MW];                   // west-face flux (f0, f1L, f2) of every thread, by row parity
    T er[3][MARCH_MAX_R];             // east-edge face of the strip for every row of the chunk
    T sw[4][MARCH_MAX_R];             // state of column x0-1 for every row of the chunk
    T red[32];
};

// HLLC/HLL flux on hydrostatically reconstructed states, from (eta, u_n, u_t, z) of both sides.
// Same flux as riemann()+face_flux() of flood.cuh, rewritten so that
//  - only eta = h + z and z are needed (h* = max(0, eta - max(zL, zR))),
//  - the dry-bed wave speeds come out of the two-rarefaction formulas by substituting
//    u_dry := u_wet -/+ 2 c_wet for the dry side (identical values, no selects on s_L, s_R),
//  - the per-side pressure corrections are folded in: f1L = F1 - g hL*^2/2, f1R = f1L - de.
// Equal reconstructed states give f0 = 0 and f1L = f1R = 0 exactly (lake at rest).
template <typename T, bool SOLID, bool VOTE>
__device__ __forceinline__ void face_eta(T g, T etaL, T uL, T vL, T zL, T etaR, T uR, T vR, T zR,
                                         T &f0, T &f1L, T &f1R, T &f2)
{
    if (SOLID) {                      // wall ghost of the other side (C13, C16)
        const bool sl = is_solid(zL), sr = is_solid(zR);
        if (sl) { etaL = etaR; uL = -uR; vL = vR; zL = zR; }
        if (sr) { etaR = etaL; uR = -uL; vR = vL; zR = zL; }
    }
    const T zf = fmax(zL, zR);
    const T hL = fmax(T(0), etaL - zf);       // both solid: inf - inf = NaN -> fmax gives 0
    const T hR = fmax(T(0), etaR - zf);
    const bool wet = fmax(hL, hR) > T(0);
    if (VOTE ? !__any_sync(0xffffffffu, wet) : !wet) { f0 = f1L = f1R = f2 = T(0); return; }
    const T ghL = g * hL, ghR = g * hR;
    const T cL = fast_sqrt(ghL), cR = fast_sqrt(ghR);
    const T uLe = hL > T(0) ? uL : uR - T(2) * cR;
    const T uRe = hR > T(0) ? uR : uL + T(2) * cL;
    const T us = T(0.5) * (uLe + uRe) + (cL - cR);
    const T cs = T(0.5) * (cL + cR) + T(0.25) * (uLe - uRe);
    const T sL = fmin(fmin(uLe - cL, us - cs), T(0));
    const T sR = fmax(fmax(uRe + cR, us + cs), T(0));
    const T qL = hL * uLe, qR = hR * uRe;
    const T mL = qL * uLe, mR = qR * uRe;
    const T de = T(0.5) * (ghR * hR - ghL * hL);
    const T w = -sL * fast_rcp(fmax(sR - sL, T(1e-30)));
    const T dq = qR - qL;
    f0 = qL + w * (dq - sR * (hR - hL));
    f1L = mL + w * (((mR - mL) + de) - sR * dq);
    f1R = f1L - de;
    f2 = f0 * (f0 >= T(0) ? vL : vR);
}

// clamp (C12), Manning friction (C6), wave speed of the new state for the CFL reduction
template <typename T>
__device__ __forceinline__ void finish_hat(const FloodArgs<T> &a, T dt, T &hn, T &qxn, T &qyn, T n0, int np, T &lam)
{
    if (hn < T(0)) {
        atomicAdd(&a.ctl->clamped_volume, (double)(-hn) * (double)a.cell_area);
        atomicAdd(&a.ctl->neg_clamps, 1ull);
        hn = T(0);
    }
    if (hn > a.h_dry) {
        const T n = a.couple ? n0 * (T(1) + T(min(np, a.n_cap))) : n0;
        const T D = T(1) + dt * a.g * n * n * fast_sqrt(qxn * qxn + qyn * qyn) * pow_m73(hn);
        const T rD = fast_rcp(D);
        qxn *= rD; qyn *= rD;
        const T rh = fast_rcp(hn), c = fast_sqrt(a.g * hn);
        lam = fmax(lam, fmax((fabs(qxn * rh) + c) * a.inv_dx, (fabs(qyn * rh) + c) * a.inv_dy));
    } else { qxn = T(0); qyn = T(0); }
}

template <typename T> struct Raw4 { T h, qx, qy, z; };

template <typename T, bool GEN>
__device__ __forceinline__ Raw4<T> march_load(const T *__restrict__ H, const T *__restrict__ QX,
                                              const T *__restrict__ QY, const T *__restrict__ Z,
                                              int i, int j, int nx, int ny)
{
    Raw4<T> r;
    if (GEN && (i < 0 || i >= nx || j < 0 || j >= ny)) { r.h = r.qx = r.qy = T(0); r.z = solid_z<T>(); return r; }
    const size_t c = (size_t)j * nx + i;
    r.h = H[c]; r.qx = QX[c]; r.qy = QY[c]; r.z = Z[c];
    return r;
}

// raw conserved -> (eta, u, v); a solid cell has h = 0, u = v = 0, eta = +inf
template <typename T, bool GEN>
__device__ __forceinline__ void march_prims(Raw4<T> &r, T h_dry, T &eta, T &u, T &v)
{
    if (GEN && is_solid(r.z)) { r.h = r.qx = r.qy = T(0); }
    primitives(r.h, r.qx, r.qy, h_dry, u, v);
    eta = r.h + r.z;
}

template <typename T, bool GEN>
__device__ __forceinline__ T march_chunk(const FloodArgs<T> &a, MarchSmem<T> &s, int x0, int y0, int R)
{
    const int tid = threadIdx.x;
    const int nx = a.nx, ny = a.ny;
    const int p = a.ctl->parity;
    const uint8_t *__restrict__ OCC = a.occ + (size_t)p * a.occ_stride;
    const T *__restrict__ H = a.h[p], *__restrict__ QX = a.qx[p], *__restrict__ QY = a.qy[p];
    const T *__restrict__ Z = a.zs;
    T *__restrict__ Ho = a.h[p ^ 1], *__restrict__ QXo = a.qx[p ^ 1], *__restrict__ QYo = a.qy[p ^ 1];
    const T dt = (T)a.ctl->dt;
    const T qin = GEN ? (T)a.ctl->q_in : T(0);
    const T dtdx = dt * a.inv_dx, dtdy = dt * a.inv_dy;
    const T g = a.g, h_dry = a.h_dry;
    const int i = x0 + tid;
    const bool col_ok = GEN ? (i < nx) : true;
    const int y1 = min(y0 + R, ny);                    // rows [y0, y1) are owned by this chunk

    // rows y0-1 (halo), y0, y0+1 on their way
    Raw4<T> rp = march_load<T, GEN>(H, QX, QY, Z, i, y0 - 1, nx, ny);
    Raw4<T> c0 = march_load<T, GEN>(H, QX, QY, Z, i, y0, nx, ny);
    Raw4<T> c1 = march_load<T, GEN>(H, QX, QY, Z, i, min(y0 + 1, GEN ? y0 + 1 : y1), nx, ny);

    // ---- pre-pass: strip-edge data for every row of the chunk
    if (tid < R) {                                     // east-edge face between columns x0+MW-1 and x0+MW
        const int j = y0 + tid;
        T f0 = T(0), f1L = T(0), f1R, f2 = T(0);
        if (j < y1) {
            Raw4<T> l = march_load<T, GEN>(H, QX, QY, Z, x0 + MW - 1, j, nx, ny);
            Raw4<T> r = march_load<T, GEN>(H, QX, QY, Z, x0 + MW, j, nx, ny);
            T el, ul, vl, er_, ur, vr;
            march_prims<T, GEN>(l, h_dry, el, ul, vl);
            march_prims<T, GEN>(r, h_dry, er_, ur, vr);
            face_eta<T, GEN, false>(g, el, ul, vl, l.z, er_, ur, vr, r.z, f0, f1L, f1R, f2);
        }
        s.er[0][tid] = f0; s.er[1][tid] = f1L; s.er[2][tid] = f2;
    } else if (tid >= MARCH_MAX_R && tid < MARCH_MAX_R + R) {     // state of column x0-1
        const int k = tid - MARCH_MAX_R, j = y0 + k;
        Raw4<T> l = march_load<T, true>(H, QX, QY, Z, x0 - 1, min(j, ny - 1), nx, ny);
        T el, ul, vl;
        march_prims<T, true>(l, h_dry, el, ul, vl);
        s.sw[0][k] = el; s.sw[1][k] = ul; s.sw[2][k] = vl; s.sw[3][k] = l.z;
    }

    // halo row y0-1 becomes "prev"
    T eta_p, u_p, v_p, z_p;
    march_prims<T, GEN>(rp, h_dry, eta_p, u_p, v_p);
    z_p = rp.z;
    T ah = T(0), ax = T(0), ay = T(0), n0_p = T(0);    // accumulators of the previous (owned) row
    int occ_p = 0;
    T lam = T(0);

    for (int jj = y0; jj <= y1; ++jj) {
        Raw4<T> cur = c0;
        c0 = c1;
        c1 = march_load<T, GEN>(H, QX, QY, Z, i, GEN ? jj + 2 : min(jj + 2, y1), nx, ny);
        T eta, u, v;
        march_prims<T, GEN>(cur, h_dry, eta, u, v);
        const int b = jj & 1;
        s.st[b][0][tid] = eta; s.st[b][1][tid] = u; s.st[b][2][tid] = v; s.st[b][3][tid] = cur.z;
        T n0_c = T(0); int occ_c = 0;
        if (jj < y1 && col_ok) {
            const size_t c = (size_t)jj * nx + i;
            n0_c = a.n0[c];
            occ_c = a.couple ? (int)OCC[c] : 0;
        }
        __syncthreads();

        // south face of the current row = north face of the previous one (normal velocity v)
        T g0, g1L, g1R, g2;
        face_eta<T, GEN, true>(g, eta_p, v_p, u_p, z_p, eta, v, u, cur.z, g0, g1L, g1R, g2);

        if (jj > y0) {                                 // finish row jj-1
            const int j = jj - 1, bp = b ^ 1;
            const T *fe = (tid == MW - 1) ? &s.er[0][j - y0] : &s.fx[bp][0][tid + 1];
            const int stride = (tid == MW - 1) ? MARCH_MAX_R : MW;
            T hn = ah - dtdx * fe[0] - dtdy * g0;
            T qxn = ax - dtdx * fe[stride] - dtdy * g2;
            T qyn = ay - dtdx * fe[2 * stride] - dtdy * g1L;
            if (GEN) {
                if (i == nx - 1) hn += dtdx * qin * T(a.inflow[1][j]);
                if (j == ny - 1 && col_ok) hn += dtdy * qin * T(a.inflow[3][i]);
            }
            if (GEN && is_solid(z_p)) { hn = qxn = qyn = T(0); }
            else finish_hat(a, dt, hn, qxn, qyn, n0_p, occ_p, lam);
            if (col_ok) {
                const size_t c = (size_t)j * nx + i;
                Ho[c] = hn; QXo[c] = qxn; QYo[c] = qyn;
            }
        }
        if (jj < y1) {                                 // enter row jj: west face, start its accumulators
            const T *sl = (tid == 0) ? &s.sw[0][jj - y0] : &s.st[b][0][tid - 1];
            const int stride = (tid == 0) ? MARCH_MAX_R : MW;
            T f0, f1L, f1R, f2;
            face_eta<T, GEN, true>(g, sl[0], sl[stride], sl[2 * stride], sl[3 * stride], eta, u, v, cur.z, f0, f1L, f1R, f2);
            s.fx[b][0][tid] = f0; s.fx[b][1][tid] = f1L; s.fx[b][2][tid] = f2;
            ah = cur.h + dtdx * f0 + dtdy * g0;
            ax = cur.qx + dtdx * f1R + dtdy * g2;
            ay = cur.qy + dtdx * f2 + dtdy * g1R;
            if (GEN) {
                if (i == 0) ah += dtdx * qin * T(a.inflow[0][jj]);
                if (jj == 0 && col_ok) ah += dtdy * qin * T(a.inflow[2][i]);
            }
        }
        eta_p = eta; u_p = u; v_p = v; z_p = cur.z; n0_p = n0_c; occ_p = occ_c;
    }
    return lam;
}

template <typename T>
__global__ void __launch_bounds__(MW, sizeof(T) == 4 ? 4 : 2) flood_march_kernel(FloodArgs<T> a)
{
    pdl_enter();
    __shared__ MarchSmem<T> s;
    if (a.ctl->halt) return;
    const int x0 = blockIdx.x * MW, y0 = blockIdx.y * a.R;
    const bool gen = a.chunk_flag[blockIdx.y * gridDim.x + blockIdx.x] != 0;
    T lam = gen ? march_chunk<T, true>(a, s, x0, y0, a.R) : march_chunk<T, false>(a, s, x0, y0, a.R);
    const int tid = threadIdx.x;
    for (int o = 16; o > 0; o >>= 1) lam = fmax(lam, __shfl_xor_sync(0xffffffffu, lam, o));
    __syncthreads();
    if ((tid & 31) == 0) s.red[tid >> 5] = lam;
    __syncthreads();
    if (tid < 32) {
        T m = tid < MW / 32 ? s.red[tid] : T(0);
        for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (tid == 0 && m > T(0)) atomic_max_lambda(a.ctl, (double)m);
    }
}

// Which path a chunk takes: 1 = it touches the domain edge and its strip sticks out of the domain
// (general path: bounds checks, wall ghosts, inflow); 3 = it touches the domain edge, strip inside
// (variant 4: TMA path with ghost rows; variants 2 and 3 treat it like 1); 2 = interior, but a solid cell lies in it or in its one-cell halo (the row-marching
// kernels with wall-ghost selects; variants 2 and 3 treat it like 1); 0 = interior, no solid.
// One CTA per chunk; rerun whenever the bed array is rewritten.
template <typename T>
__global__ void flood_chunk_flags_kernel(const T *__restrict__ zs, int nx, int ny, int R, uint8_t *flag)
{
    const int x0 = blockIdx.x * MW, y0 = blockIdx.y * R;
    const int edge = (x0 == 0) || (y0 == 0) || (x0 + MW >= nx) || (y0 + R >= ny);
    int solid = 0;
    if (!edge) {
        const int w = MW + 2, n = w * (R + 2);
        for (int k = threadIdx.x; k < n; k += blockDim.x) {
            const int i = x0 - 1 + k % w, j = y0 - 1 + k / w;
            if (is_solid(zs[(size_t)j * nx + i])) solid = 1;
        }
    }
    solid = __syncthreads_or(solid);
    if (threadIdx.x == 0) flag[blockIdx.y * gridDim.x + blockIdx.x] = (uint8_t)(edge ? (x0 + MW <= nx ? 3 : 1) : solid ? 2 : 0);
}

}  // namespace fp
