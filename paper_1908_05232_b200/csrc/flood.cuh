// flood.cuh -- step (F)+(T) of include/floodped.h: the flood-cell update, Eq. (2) of the paper
// (P:L105), with the CFL reduction for the next step fused in.
//
//   U^{n+1} = U^n - dt/dx (F_E - F_W) - dt/dy (G_N - G_S) + S
//
// Face fluxes: HLLC on hydrostatically reconstructed states (C2-C4; the scheme the
// paper cites at P:L97, L108); bed slope folded into per-side pressure corrections; Manning
// friction pointwise semi-implicit (C6); wall ghosts at the domain edge and at solid cells
// (C13, C16); accounted clamp of negative depth (C12).
//
// Two kernels compute the same thing:
//   flood_cell_kernel   one thread per cell, all 4 faces per cell, operands from global/L1.
//                       Simple; kept as the A/B baseline and for nx % 4 != 0.
//   flood_tile_kernel   64x16-cell tile + halo staged in shared memory as primitives, 128-bit
//                       coalesced SoA loads/stores, every face evaluated ONCE (tile-edge faces
//                       by a 9th helper warp), fluxes exchanged through shared memory.
#pragma once

#include "common.cuh"

namespace fp {

template <typename T>
struct FloodArgs {
    int nx, ny;
    T g, inv_dx, inv_dy, h_dry, cell_area;
    int couple, n_cap;
    T *h[2], *qx[2], *qy[2];          // ping-pong conserved state, SoA, row-major
    const T *zs;                      // bed elevation; +inf marks a solid cell
    const T *n0;                      // initial Manning n_M per cell
    const uint8_t *occ;               // N_p per cell (saturated at 255): buffer 0; the step at flood parity p reads occ + p * occ_stride
    size_t occ_stride;
    const uint8_t *inflow[4];         // per edge cell: number of inflow faces on that side (W,E,S,N)
    const uint8_t *chunk_flag;        // march kernels: path of every chunk (flood_chunk_flags_kernel)
    const T *ghost_zero, *ghost_inf;  // one strip-wide row of zeros / of +inf, and of zero bytes: the row beyond the
    const uint8_t *ghost_occ;         // domain edge as the TMA kernel loads it (a wall = a row of solid cells, C13)
    int R;                            // march kernel: rows per chunk
    // row slabs: the row below my first row / above my last row is the boundary row of the
    // neighbour slab, read in place -- peer memory over NVLink, or another handle on the same device.
    // [0 south | 1 north][flood parity]; null = the domain edge (wall ghost).  Kernels 0 and 4.
    const T *halo_h[2][2], *halo_qx[2][2], *halo_qy[2][2];
    const T *halo_z[2];
    uint8_t *dryseg;                  // TMA march kernel: [2][chunk rows][nsegx] dry-segment flags (see flood_tmarch_kernel); null = off
    size_t dry_stride; int nsegx;
    int open_sides;                   // bit per domain edge (W, E, S, N): open, transmissive ghost; kernels 0 and 5 only
    Ctl *ctl;
};

// D1: is the domain-edge face of cell (i, j) on `side` open?  Inflow faces stay inflow faces (C14).
template <typename T>
__device__ __forceinline__ bool open_face(const FloodArgs<T> &a, int side, int i, int j)
{
    return ((a.open_sides >> side) & 1) && a.inflow[side][side < 2 ? j : i] == 0;
}

// volume leaving through an open face this step (D1): V = V0 + inflow - outflow + clamped
template <typename T>
__device__ __forceinline__ void add_outflow(const FloodArgs<T> &a, T dt, T flux_out, T inv_len_other)
{
    // face length = cell_area * (1 / the other side's length)
    atomicAdd(&a.ctl->outflow_volume, (double)dt * (double)flux_out * ((double)a.cell_area * (double)inv_len_other));
}

// ------------------------------------------------------------------------------------------------
// HLLC flux on already reconstructed states.  Two-rarefaction wave-speed estimates with the
// dry-bed limits (C3).  The tangential momentum is upwinded with the sign of the mass flux, which
// is the sign of the contact speed s_M (same sign in every branch).
template <typename T>
__device__ __forceinline__ void riemann(T g, T hL, T uL, T vL, T hR, T uR, T vR, T &f0, T &f1, T &f2)
{
    // branch-free: selects for the dry-bed speeds, and the upwind cases fall out of clamping the
    // wave speeds (s_L <- min(s_L,0), s_R <- max(s_R,0)): w = 0 gives F_L, w = 1 gives F_R.
    const T cL = fast_sqrt(g * hL), cR = fast_sqrt(g * hR);
    const T us = T(0.5) * (uL + uR) + cL - cR;
    const T cs = T(0.5) * (cL + cR) + T(0.25) * (uL - uR);
    T sL = fmin(uL - cL, us - cs);
    T sR = fmax(uR + cR, us + cs);
    const bool dryL = hL <= T(0), dryR = hR <= T(0);
    sL = dryL ? uR - T(2) * cR : sL;  sR = dryL ? uR + cR : sR;
    sR = dryR ? uL + T(2) * cL : sR;  sL = dryR ? uL - cL : sL;
    sL = fmin(sL, T(0)); sR = fmax(sR, T(0));
    const T qL = hL * uL, qR = hR * uR;
    const T pL = qL * uL + T(0.5) * g * hL * hL;
    const T pR = qR * uR + T(0.5) * g * hR * hR;
    // HLL written around F_L: F = F_L + w [(F_R - F_L) - s_R (U_R - U_L)], w = -s_L/(s_R - s_L).
    // Equal states give F_L exactly whatever the rounding of w (lake at rest stays at rest).
    const T w = -sL * fast_rcp(fmax(sR - sL, T(1e-30)));      // s_R = s_L = 0 only if s_L = 0: w = 0
    const T dq = qR - qL;
    f0 = qL + w * (dq - sR * (hR - hL));
    f1 = pL + w * ((pR - pL) - sR * dq);
    f2 = f0 * (f0 >= T(0) ? vL : vR);
}

// One face between a left/lower cell L and a right/upper cell R given as primitives
// (h, normal velocity, tangential velocity, bed).  A solid side (z = +inf) is replaced by the
// wall ghost of the other side.  Returns mass flux f0, normal-momentum flux as seen by L (f1L)
// and by R (f1R) -- the bed-slope source is the difference -- and tangential-momentum flux f2.
template <typename T>
__device__ __forceinline__ void face_flux(T g, T hL, T unL, T utL, T zL, T hR, T unR, T utR, T zR,
                                          T &f0, T &f1L, T &f1R, T &f2)
{
    const bool sL = is_solid(zL), sR = is_solid(zR);
    if (sL) { hL = hR; unL = -unR; utL = utR; zL = zR; }
    if (sR) { hR = hL; unR = -unL; utR = utL; zR = zL; }
    const T zf = fmax(zL, zR);
    const T hLs = fmax(T(0), (hL + zL) - zf);
    const T hRs = fmax(T(0), (hR + zR) - zf);
    if ((hLs <= T(0) && hRs <= T(0)) || (sL && sR)) { f0 = f1L = f1R = f2 = T(0); return; }
    T f1;
    riemann(g, hLs, unL, utL, hRs, unR, utR, f0, f1, f2);
    f1L = f1 - T(0.5) * g * hLs * hLs;
    f1R = f1 - T(0.5) * g * hRs * hRs;
}

template <typename T>
__device__ __forceinline__ void primitives(T h, T qx, T qy, T h_dry, T &u, T &v)
{
    if (h > h_dry) { const T r = fast_rcp(h); u = qx * r; v = qy * r; }
    else { u = T(0); v = T(0); }
}

// Everything after the four faces: Eq. (2), clamp, friction, wave speed of the new state.
template <typename T>
__device__ __forceinline__ void finish_cell(const FloodArgs<T> &a, T dt, T h, T qx, T qy,
                                            T dF0, T dF1, T dF2, T dG0, T dG1, T dG2,
                                            T n0, int np, T &hn, T &qxn, T &qyn, T &lam)
{
    const T dtdx = dt * a.inv_dx, dtdy = dt * a.inv_dy;
    hn  = h  - dtdx * dF0 - dtdy * dG0;
    qxn = qx - dtdx * dF1 - dtdy * dG1;
    qyn = qy - dtdx * dF2 - dtdy * dG2;
    if (hn < T(0)) {                                   // C12: rare, accounted
        atomicAdd(&a.ctl->clamped_volume, (double)(-hn) * (double)a.cell_area);
        atomicAdd(&a.ctl->neg_clamps, 1ull);
        hn = T(0);
    }
    lam = T(0);
    if (hn > a.h_dry) {
        const T n = a.couple ? n0 * (T(1) + T(min(np, a.n_cap))) : n0;
        const T D = T(1) + dt * a.g * n * n * fast_sqrt(qxn * qxn + qyn * qyn) * pow_m73(hn);
        const T rD = fast_rcp(D);
        qxn *= rD; qyn *= rD;
        const T rh = fast_rcp(hn), c = fast_sqrt(a.g * hn);
        lam = fmax((fabs(qxn * rh) + c) * a.inv_dx, (fabs(qyn * rh) + c) * a.inv_dy);
    } else { qxn = T(0); qyn = T(0); }
}

// block-wide max of lam -> one atomic per block
template <typename T>
__device__ __forceinline__ void block_max_lambda(Ctl *ctl, T lam, T *warp_scratch /* [32] shared */)
{
    for (int o = 16; o > 0; o >>= 1) lam = fmax(lam, __shfl_xor_sync(0xffffffffu, lam, o));
    const int tid = threadIdx.y * blockDim.x + threadIdx.x;
    const int nw = (blockDim.x * blockDim.y + 31) >> 5;
    if ((tid & 31) == 0) warp_scratch[tid >> 5] = lam;
    __syncthreads();
    if (tid < 32) {
        T m = tid < nw ? warp_scratch[tid] : T(0);
        for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (tid == 0 && m > T(0)) atomic_max_lambda(ctl, (double)m);
    }
}

// ------------------------------------------------------------------------------------------------
// Variant 0: one thread per cell.
template <typename T>
__global__ void __launch_bounds__(256) flood_cell_kernel(FloodArgs<T> a)
{
    pdl_enter();
    __shared__ T red[32];
    if (a.ctl->halt) return;
    const int p = a.ctl->parity;
    const uint8_t *__restrict__ OCC = a.occ + (size_t)p * a.occ_stride;
    const T *__restrict__ H = a.h[p], *__restrict__ QX = a.qx[p], *__restrict__ QY = a.qy[p];
    const T *__restrict__ Z = a.zs;
    const T dt = (T)a.ctl->dt, qin = (T)a.ctl->q_in;
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
    T lam = T(0);
    if (i < a.nx && j < a.ny) {
        const int c = j * a.nx + i;
        const T z = Z[c];
        T hn = T(0), qxn = T(0), qyn = T(0);
        if (!is_solid(z)) {
            const T h = H[c], qx = QX[c], qy = QY[c];
            T u, v; primitives(h, qx, qy, a.h_dry, u, v);
            const bool oW = i == 0 && open_face(a, 0, i, j), oE = i == a.nx - 1 && open_face(a, 1, i, j);
            const bool oS = j == 0 && open_face(a, 2, i, j), oN = j == a.ny - 1 && open_face(a, 3, i, j);
            auto nb = [&](int ii, int jj, bool open, T &hk, T &uk, T &vk, T &zk) {
                zk = solid_z<T>(); hk = uk = vk = T(0);
                if (ii >= 0 && jj >= 0 && ii < a.nx && jj < a.ny) {
                    const int k = jj * a.nx + ii;
                    zk = Z[k];
                    if (!is_solid(zk)) { hk = H[k]; primitives(hk, QX[k], QY[k], a.h_dry, uk, vk); }
                } else if ((jj < 0 || jj >= a.ny) && ii >= 0 && ii < a.nx && a.halo_z[jj < 0 ? 0 : 1]) {
                    const int sd = jj < 0 ? 0 : 1;                          // the neighbour slab's boundary row (8f-4)
                    zk = a.halo_z[sd][ii];
                    if (!is_solid(zk)) { hk = a.halo_h[sd][p][ii]; primitives(hk, a.halo_qx[sd][p][ii], a.halo_qy[sd][p][ii], a.h_dry, uk, vk); }
                } else if (open) { hk = h; uk = u; vk = v; zk = z; }       // transmissive ghost (D1)
            };
            T hk, uk, vk, zk, f1L, f1R;
            T FE0, FE1, FE2, FW0, FW1, FW2, GN0, GN1, GN2, GS0, GS1, GS2;
            nb(i + 1, j, oE, hk, uk, vk, zk);
            face_flux(a.g, h, u, v, z, hk, uk, vk, zk, FE0, f1L, f1R, FE2); FE1 = f1L;
            nb(i - 1, j, oW, hk, uk, vk, zk);
            face_flux(a.g, hk, uk, vk, zk, h, u, v, z, FW0, f1L, f1R, FW2); FW1 = f1R;
            nb(i, j + 1, oN, hk, uk, vk, zk);
            face_flux(a.g, h, v, u, z, hk, vk, uk, zk, GN0, f1L, f1R, GN1); GN2 = f1L;
            nb(i, j - 1, oS, hk, uk, vk, zk);
            face_flux(a.g, hk, vk, uk, zk, h, v, u, z, GS0, f1L, f1R, GS1); GS2 = f1R;
            if (i == 0) FW0 += qin * T(a.inflow[0][j]);
            if (i == a.nx - 1) FE0 -= qin * T(a.inflow[1][j]);
            if (j == 0) GS0 += qin * T(a.inflow[2][i]);
            if (j == a.ny - 1) GN0 -= qin * T(a.inflow[3][i]);
            if (oE) add_outflow(a, dt, FE0, a.inv_dx);
            if (oW) add_outflow(a, dt, -FW0, a.inv_dx);
            if (oN) add_outflow(a, dt, GN0, a.inv_dy);
            if (oS) add_outflow(a, dt, -GS0, a.inv_dy);
            finish_cell(a, dt, h, qx, qy, FE0 - FW0, FE1 - FW1, FE2 - FW2, GN0 - GS0, GN1 - GS1, GN2 - GS2,
                        a.n0[c], (int)OCC[c], hn, qxn, qyn, lam);
        }
        a.h[p ^ 1][c] = hn; a.qx[p ^ 1][c] = qxn; a.qy[p ^ 1][c] = qyn;
    }
    block_max_lambda(a.ctl, lam, red);
}

// ------------------------------------------------------------------------------------------------
// Variant 1: tiled.  Block = 8 main warps (16 x 16 threads, 4 x-consecutive cells per thread
// -> 64 x 16 cells) + 1 helper warp.  Shared memory, all SoA:
//   prim[4][TY+2][PW]      h, u, v, z of tile + halo ring (z = +inf: solid or outside)
//   xfl[3][TY][TXQ+1]      (f0, f1L, f2) of the WEST face of each thread's first cell; slot TXQ of
//                          each row = the tile's east-edge face (helper warp)
//   yfl[3][TY+1][TX]       (f0, f1L, f2) of the SOUTH face of every cell; row TY = the tile's
//                          north-edge faces (helper warp)
// A thread needs f1R of its own west/south faces only, so f1R never leaves registers.
constexpr int TX = 64, TY = 16, TXQ = TX / 4;
constexpr int PW = TX + 8;            // prim row pitch: x = -1 sits at column 3, x = 0 at column 4 (16 B aligned)
constexpr int FLOOD_TILE_THREADS = TXQ * TY + 32;

template <typename T>
struct TileSmem {
    T prim[4][TY + 2][PW];
    T xfl[3][TY][TXQ + 1];
    T yfl[3][TY + 1][TX];
    T red[32];
};

template <typename T>
__global__ void __launch_bounds__(FLOOD_TILE_THREADS, sizeof(T) == 4 ? 3 : 1) flood_tile_kernel(FloodArgs<T> a)
{
    pdl_enter();
    extern __shared__ __align__(32) unsigned char smem_raw[];
    TileSmem<T> &s = *reinterpret_cast<TileSmem<T> *>(smem_raw);
    if (a.ctl->halt) return;
    const int p = a.ctl->parity;
    const uint8_t *__restrict__ OCC = a.occ + (size_t)p * a.occ_stride;
    const T *__restrict__ H = a.h[p], *__restrict__ QX = a.qx[p], *__restrict__ QY = a.qy[p];
    const T *__restrict__ Z = a.zs;
    const T dt = (T)a.ctl->dt, qin = (T)a.ctl->q_in;
    const int tid = threadIdx.x;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
    const bool helper = tid >= TXQ * TY;
    const int tx = tid % TXQ, ty = tid / TXQ;          // main threads
    const int gx = x0 + 4 * tx, gy = y0 + ty;
    const bool inside = !helper && gx < a.nx && gy < a.ny;   // nx % 4 == 0: a quad is all in or all out

    // ---- phase 1: load tile + halo, convert to primitives, stage in shared memory
    Vec4<T> h4, qx4, qy4, z4, u4, v4;
    auto put = [&](int r, int col, T hh, T uu, T vv, T zz) {
        s.prim[0][r][col] = hh; s.prim[1][r][col] = uu; s.prim[2][r][col] = vv; s.prim[3][r][col] = zz;
    };
    auto load_cell = [&](int ii, int jj, T &hh, T &uu, T &vv, T &zz) {
        hh = uu = vv = T(0); zz = solid_z<T>();
        if (ii >= 0 && jj >= 0 && ii < a.nx && jj < a.ny) {
            const int k = jj * a.nx + ii;
            zz = Z[k];
            if (!is_solid(zz)) { hh = H[k]; primitives(hh, QX[k], QY[k], a.h_dry, uu, vv); }
        }
    };
    if (!helper) {
        if (inside) {
            const size_t c = (size_t)gy * a.nx + gx;
            h4 = *reinterpret_cast<const Vec4<T> *>(H + c);
            qx4 = *reinterpret_cast<const Vec4<T> *>(QX + c);
            qy4 = *reinterpret_cast<const Vec4<T> *>(QY + c);
            z4 = *reinterpret_cast<const Vec4<T> *>(Z + c);
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                if (is_solid(z4.v[k])) { h4.v[k] = qx4.v[k] = qy4.v[k] = T(0); }
                primitives(h4.v[k], qx4.v[k], qy4.v[k], a.h_dry, u4.v[k], v4.v[k]);
            }
        } else {
#pragma unroll
            for (int k = 0; k < 4; ++k) { h4.v[k] = qx4.v[k] = qy4.v[k] = u4.v[k] = v4.v[k] = T(0); z4.v[k] = solid_z<T>(); }
        }
        *reinterpret_cast<Vec4<T> *>(&s.prim[0][ty + 1][4 + 4 * tx]) = h4;
        *reinterpret_cast<Vec4<T> *>(&s.prim[1][ty + 1][4 + 4 * tx]) = u4;
        *reinterpret_cast<Vec4<T> *>(&s.prim[2][ty + 1][4 + 4 * tx]) = v4;
        *reinterpret_cast<Vec4<T> *>(&s.prim[3][ty + 1][4 + 4 * tx]) = z4;
        // halo: south and north rows (64 + 64 cells) by the first 128 threads, west/east columns
        // (16 + 16 cells) by the next 32
        T hh, uu, vv, zz;
        if (tid < 2 * TX) {
            const int xx = tid % TX, top = tid / TX;
            load_cell(x0 + xx, top ? y0 + TY : y0 - 1, hh, uu, vv, zz);
            put(top ? TY + 1 : 0, 4 + xx, hh, uu, vv, zz);
        } else if (tid < 2 * TX + 2 * TY) {
            const int yy = (tid - 2 * TX) % TY, right = (tid - 2 * TX) / TY;
            load_cell(right ? x0 + TX : x0 - 1, y0 + yy, hh, uu, vv, zz);
            put(yy + 1, right ? 4 + TX : 3, hh, uu, vv, zz);
        }
    }
    __syncthreads();

    // ---- phase 2: every face once
    T fw0[4], fw1L[4], fw1R[4], fw2[4];     // west faces of my 4 cells
    T fs0[4], fs1R[4], fs2[4];              // south faces of my 4 cells (f1L goes to shared)
    if (!helper) {
        // west neighbour of my first cell comes from shared memory (column 4*tx+3)
        T hl = s.prim[0][ty + 1][4 * tx + 3], ul = s.prim[1][ty + 1][4 * tx + 3];
        T vl = s.prim[2][ty + 1][4 * tx + 3], zl = s.prim[3][ty + 1][4 * tx + 3];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            face_flux(a.g, hl, ul, vl, zl, h4.v[k], u4.v[k], v4.v[k], z4.v[k], fw0[k], fw1L[k], fw1R[k], fw2[k]);
            hl = h4.v[k]; ul = u4.v[k]; vl = v4.v[k]; zl = z4.v[k];
        }
        s.xfl[0][ty][tx] = fw0[0]; s.xfl[1][ty][tx] = fw1L[0]; s.xfl[2][ty][tx] = fw2[0];
        const Vec4<T> hs = *reinterpret_cast<const Vec4<T> *>(&s.prim[0][ty][4 + 4 * tx]);
        const Vec4<T> us = *reinterpret_cast<const Vec4<T> *>(&s.prim[1][ty][4 + 4 * tx]);
        const Vec4<T> vs = *reinterpret_cast<const Vec4<T> *>(&s.prim[2][ty][4 + 4 * tx]);
        const Vec4<T> zs = *reinterpret_cast<const Vec4<T> *>(&s.prim[3][ty][4 + 4 * tx]);
        Vec4<T> g0, g1, g2;
#pragma unroll
        for (int k = 0; k < 4; ++k) {       // y faces: normal velocity is v, tangential u
            face_flux(a.g, hs.v[k], vs.v[k], us.v[k], zs.v[k], h4.v[k], v4.v[k], u4.v[k], z4.v[k],
                      fs0[k], g1.v[k], fs1R[k], fs2[k]);
            g0.v[k] = fs0[k]; g2.v[k] = fs2[k];
        }
        *reinterpret_cast<Vec4<T> *>(&s.yfl[0][ty][4 * tx]) = g0;
        *reinterpret_cast<Vec4<T> *>(&s.yfl[1][ty][4 * tx]) = g1;
        *reinterpret_cast<Vec4<T> *>(&s.yfl[2][ty][4 * tx]) = g2;
    } else {
        // helper warp: TY east-edge faces, then TX north-edge faces
        const int l = tid - TXQ * TY;
        for (int f = l; f < TY + TX; f += 32) {
            T f0, f1L, f1R, f2;
            if (f < TY) {
                const int r = f + 1;
                face_flux(a.g, s.prim[0][r][3 + TX], s.prim[1][r][3 + TX], s.prim[2][r][3 + TX], s.prim[3][r][3 + TX],
                          s.prim[0][r][4 + TX], s.prim[1][r][4 + TX], s.prim[2][r][4 + TX], s.prim[3][r][4 + TX],
                          f0, f1L, f1R, f2);
                s.xfl[0][f][TXQ] = f0; s.xfl[1][f][TXQ] = f1L; s.xfl[2][f][TXQ] = f2;
            } else {
                const int col = 4 + (f - TY);
                face_flux(a.g, s.prim[0][TY][col], s.prim[2][TY][col], s.prim[1][TY][col], s.prim[3][TY][col],
                          s.prim[0][TY + 1][col], s.prim[2][TY + 1][col], s.prim[1][TY + 1][col], s.prim[3][TY + 1][col],
                          f0, f1L, f1R, f2);
                s.yfl[0][TY][f - TY] = f0; s.yfl[1][TY][f - TY] = f1L; s.yfl[2][TY][f - TY] = f2;
            }
        }
    }
    __syncthreads();

    // ---- phase 3: Eq. (2), friction, CFL
    T lam = T(0);
    if (inside) {
        const size_t c = (size_t)gy * a.nx + gx;
        const Vec4<T> n4 = *reinterpret_cast<const Vec4<T> *>(a.n0 + c);
        const uchar4 o4 = *reinterpret_cast<const uchar4 *>(OCC + c);
        const int occ[4] = {o4.x, o4.y, o4.z, o4.w};
        const T fe0 = s.xfl[0][ty][tx + 1], fe1L = s.xfl[1][ty][tx + 1], fe2 = s.xfl[2][ty][tx + 1];
        const Vec4<T> n0v = *reinterpret_cast<const Vec4<T> *>(&s.yfl[0][ty + 1][4 * tx]);
        const Vec4<T> n1v = *reinterpret_cast<const Vec4<T> *>(&s.yfl[1][ty + 1][4 * tx]);
        const Vec4<T> n2v = *reinterpret_cast<const Vec4<T> *>(&s.yfl[2][ty + 1][4 * tx]);
        Vec4<T> ho, qxo, qyo;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            T FW0 = fw0[k], FE0 = k < 3 ? fw0[k + 1] : fe0;
            const T FE1 = k < 3 ? fw1L[k + 1] : fe1L, FE2 = k < 3 ? fw2[k + 1] : fe2;
            T GS0 = fs0[k], GN0 = n0v.v[k];
            const int i = gx + k;
            if (i == 0) FW0 += qin * T(a.inflow[0][gy]);
            if (i == a.nx - 1) FE0 -= qin * T(a.inflow[1][gy]);
            if (gy == 0) GS0 += qin * T(a.inflow[2][i]);
            if (gy == a.ny - 1) GN0 -= qin * T(a.inflow[3][i]);
            T hn = T(0), qxn = T(0), qyn = T(0), l = T(0);
            if (!is_solid(z4.v[k]))
                finish_cell(a, dt, h4.v[k], qx4.v[k], qy4.v[k],
                            FE0 - FW0, FE1 - fw1R[k], FE2 - fw2[k],
                            GN0 - GS0, n2v.v[k] - fs2[k], n1v.v[k] - fs1R[k],
                            n4.v[k], occ[k], hn, qxn, qyn, l);
            ho.v[k] = hn; qxo.v[k] = qxn; qyo.v[k] = qyn;
            lam = fmax(lam, l);
        }
        *reinterpret_cast<Vec4<T> *>(a.h[p ^ 1] + c) = ho;
        *reinterpret_cast<Vec4<T> *>(a.qx[p ^ 1] + c) = qxo;
        *reinterpret_cast<Vec4<T> *>(a.qy[p ^ 1] + c) = qyo;
    }
    // block max (1-D block)
    for (int o = 16; o > 0; o >>= 1) lam = fmax(lam, __shfl_xor_sync(0xffffffffu, lam, o));
    if ((tid & 31) == 0) s.red[tid >> 5] = lam;
    __syncthreads();
    if (tid < 32) {
        T m = tid < FLOOD_TILE_THREADS / 32 ? s.red[tid] : T(0);
        for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (tid == 0 && m > T(0)) atomic_max_lambda(a.ctl, (double)m);
    }
}

// ------------------------------------------------------------------------------------------------
// lambda of an existing state (first dt at create, and after the test hooks re-inject state)
template <typename T>
__global__ void flood_lambda_kernel(FloodArgs<T> a)
{
    __shared__ T red[32];
    const int p = a.ctl->parity;
    const uint8_t *__restrict__ OCC = a.occ + (size_t)p * a.occ_stride;
    T lam = T(0);
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < (size_t)a.nx * a.ny;
         c += (size_t)gridDim.x * blockDim.x) {
        const T h = a.h[p][c];
        if (!is_solid(a.zs[c]) && h > a.h_dry) {
            const T u = a.qx[p][c] / h, v = a.qy[p][c] / h, cc = real_sqrt(a.g * h);
            lam = fmax(lam, fmax((fabs(u) + cc) * a.inv_dx, (fabs(v) + cc) * a.inv_dy));
        }
    }
    block_max_lambda(a.ctl, lam, red);
}

// u, v, HR = (V + 0.5) h for sim_read_flood (C8)
template <typename T>
__global__ void flood_derive_kernel(FloodArgs<T> a, T *u, T *v, T *hr)
{
    const int p = a.ctl->parity;
    const uint8_t *__restrict__ OCC = a.occ + (size_t)p * a.occ_stride;
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < (size_t)a.nx * a.ny;
         c += (size_t)gridDim.x * blockDim.x) {
        const T h = a.h[p][c];
        T uu = T(0), vv = T(0), r = T(0);
        if (h > a.h_dry) {
            uu = div_rn(a.qx[p][c], h); vv = div_rn(a.qy[p][c], h);
            r = mul_rn(add_rn(fmax(fabs(uu), fabs(vv)), T(0.5)), h);
        }
        if (u) u[c] = uu;
        if (v) v[c] = vv;
        if (hr) hr[c] = r;
    }
}

// Bed for sim_read_flood: the device keeps z = +inf in solid cells (R3); the caller gets the
// elevation the cell was created with.
template <typename T>
__global__ void flood_bed_kernel(const T *__restrict__ zs, const T *__restrict__ z0, size_t n, T *out)
{
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < n; c += (size_t)gridDim.x * blockDim.x)
        out[c] = is_solid(zs[c]) ? z0[c] : zs[c];
}

// After a state re-injection (sim_write_flood): bed with the solid cells marked (z given: new bed;
// else keep), and no water in solid cells (C16).
template <typename T>
__global__ void flood_inject_kernel(T *h, T *qx, T *qy, T *zs, const T *z_new, size_t n)
{
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < n; c += (size_t)gridDim.x * blockDim.x) {
        const bool solid = is_solid(zs[c]);            // solid cells are the cells with z = +inf, for good (R3)
        if (z_new) zs[c] = solid ? solid_z<T>() : z_new[c];
        if (solid) { h[c] = T(0); qx[c] = T(0); qy[c] = T(0); }
    }
}

// volume (fp64), max h, max HR, non-finite count: two-stage reduction into out[4]
template <typename T>
__global__ void flood_stats_kernel(FloodArgs<T> a, double *out /* volume, max_h, max_hr, n_bad */)
{
    __shared__ double sv[32], sh[32], sr[32], sb[32];
    const int p = a.ctl->parity;
    const uint8_t *__restrict__ OCC = a.occ + (size_t)p * a.occ_stride;
    double vol = 0, mh = 0, mr = 0, bad = 0;
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < (size_t)a.nx * a.ny;
         c += (size_t)gridDim.x * blockDim.x) {
        if (is_solid(a.zs[c])) continue;
        const T h = a.h[p][c];
        if (!isfinite((double)h) || !isfinite((double)a.qx[p][c]) || !isfinite((double)a.qy[p][c])) { bad += 1; continue; }
        vol += (double)h;
        mh = fmax(mh, (double)h);
        if (h > a.h_dry) {                            // HR = (V + 0.5) h in the storage precision
            const T u = div_rn(a.qx[p][c], h), v = div_rn(a.qy[p][c], h);
            mr = fmax(mr, (double)mul_rn(add_rn(fmax(fabs(u), fabs(v)), T(0.5)), h));
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        vol += __shfl_xor_sync(0xffffffffu, vol, o); bad += __shfl_xor_sync(0xffffffffu, bad, o);
        mh = fmax(mh, __shfl_xor_sync(0xffffffffu, mh, o)); mr = fmax(mr, __shfl_xor_sync(0xffffffffu, mr, o));
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) { sv[w] = vol; sh[w] = mh; sr[w] = mr; sb[w] = bad; }
    __syncthreads();
    if (w == 0) {
        const int nw = blockDim.x >> 5;
        vol = l < nw ? sv[l] : 0; mh = l < nw ? sh[l] : 0; mr = l < nw ? sr[l] : 0; bad = l < nw ? sb[l] : 0;
        for (int o = 16; o > 0; o >>= 1) {
            vol += __shfl_xor_sync(0xffffffffu, vol, o); bad += __shfl_xor_sync(0xffffffffu, bad, o);
            mh = fmax(mh, __shfl_xor_sync(0xffffffffu, mh, o)); mr = fmax(mr, __shfl_xor_sync(0xffffffffu, mr, o));
        }
        if (l == 0) {
            atomicAdd(&out[0], vol * (double)a.cell_area);
            atomicMax((unsigned long long *)&out[1], (unsigned long long)__double_as_longlong(mh));
            atomicMax((unsigned long long *)&out[2], (unsigned long long)__double_as_longlong(mr));
            atomicAdd(&out[3], bad);
        }
    }
}

}  // namespace fp
