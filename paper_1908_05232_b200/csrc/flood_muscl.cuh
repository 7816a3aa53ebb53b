// flood_muscl.cuh -- second-order variant of step (F)+(T): MUSCL-Hancock.
//
// The paper's scheme is "an explicit shock-capturing scheme (Wang et al. 2011) ... reduced to
// first-order accuracy"; this is the scheme it was reduced FROM, selected with
// sim_params_t::flood_order = 2.  The paper prints none of it: the reading is DESIGN.md M1-M7,
//   M1 minmod slopes of (eta, h, qx, qy) per direction; zero where the cell or a neighbour is not
//      wet or a neighbour is a wall (first order at fronts and walls);
//   M2 face values W +- slope/2, face bed z_f = eta_f - h_f;
//   M3 Hancock half-step predictor from the cell's own face values (pressure and bed slope together
//      as g hbar d eta: still water does not move), depth clamped at 0;
//   M4 one HLLC flux per face on hydrostatically reconstructed predicted face states
//      (the same riemann() as the first-order kernels); momentum flux seen by a cell
//      F1 - g h*^2/2 + g h_f^2/2;
//   M5 centred bed-slope source g (h_W + h_E)(z_W - z_E) / 2 dx of the cell's own face values;
//   M6 update, inflow, clamp, friction, M7 CFL as in the first-order step (finish_cell()).
//
// Kernel: a CTA of 32 x 8 threads owns a tile of 32 x 8 cells.
//   phase 1  (h, qx, qy, z) of the tile + a halo of TWO cells into shared memory (z = +inf outside
//            the domain and in solid cells: a wall);
//   phase 2  predicted face values (4 faces x (h, qx, qy, z)) of the tile + a halo of ONE cell;
//   phase 3a every face of the tile once (left | right predicted face values, or the wall / transmissive
//            ghost), fluxes to shared memory;
//   phase 3b every thread: its four face fluxes, sources, finish_cell(), block-wide max of the wave speed.
// Algorithmic bytes per cell are those of the first-order step (33 B fp32); the halo-2 re-reads
// are L2 traffic.
#pragma once

#include "flood.cuh"

namespace fp {

constexpr int MTX = 32, MTY = 8;                       // tile
constexpr int MRX = MTX + 4, MRY = MTY + 4;            // raw state: halo 2
constexpr int MPX = MTX + 2, MPY = MTY + 2;            // predicted face values: halo 1

template <typename T>
struct MusclSmem {
    T raw[4][MRY][MRX];            // h, qx, qy, z
    T fv[4][4][MPY][MPX];          // predicted face values [face W,E,S,N][h, u, v, z]
    T xf[4][MTY][MTX + 1];         // x-faces of the tile: mass flux, normal momentum as seen by the left / by the right cell, tangential
    T yf[4][MTY + 1][MTX];         // y-faces likewise (lower / upper)
    uint8_t wet[MPY][MPX];         // cell wet at level n (h > h_dry), 2 = solid / outside
    T red[32];
};

template <typename T> __device__ __forceinline__ T minmod(T a, T b)
{
    if (a * b <= T(0)) return T(0);
    return fabs(a) < fabs(b) ? a : b;
}

// velocity of a face value of a WET cell: q / max(h, h_dry); a cell that is not wet has u = v = 0
template <typename T> __device__ __forceinline__ T face_vel(bool wet, T q, T h, T h_dry)
{
    return wet ? q * fast_rcp(fmax(h, h_dry)) : T(0);
}

template <typename T>
__global__ void __launch_bounds__(MTX * MTY) flood_muscl_kernel(FloodArgs<T> a)
{
    pdl_enter();
    extern __shared__ __align__(32) unsigned char smem_raw[];
    MusclSmem<T> &s = *reinterpret_cast<MusclSmem<T> *>(smem_raw);
    if (a.ctl->halt) return;
    const int p = a.ctl->parity;
    const uint8_t *__restrict__ OCC = a.occ + (size_t)p * a.occ_stride;
    const T *__restrict__ H = a.h[p], *__restrict__ QX = a.qx[p], *__restrict__ QY = a.qy[p];
    const T *__restrict__ Z = a.zs;
    const T dt = (T)a.ctl->dt, qin = (T)a.ctl->q_in;
    const int tid = threadIdx.y * MTX + threadIdx.x;
    const int x0 = blockIdx.x * MTX, y0 = blockIdx.y * MTY;

    // phase 1: raw state, halo 2
    for (int k = tid; k < MRX * MRY; k += MTX * MTY) {
        const int lx = k % MRX, ly = k / MRX, gx = x0 + lx - 2, gy = y0 + ly - 2;
        T h = T(0), qx = T(0), qy = T(0), z = solid_z<T>();
        if (gx >= 0 && gy >= 0 && gx < a.nx && gy < a.ny) {
            const int c = gy * a.nx + gx;
            z = Z[c];
            if (!is_solid(z)) { h = H[c]; qx = QX[c]; qy = QY[c]; }
        }
        s.raw[0][ly][lx] = h; s.raw[1][ly][lx] = qx; s.raw[2][ly][lx] = qy; s.raw[3][ly][lx] = z;
    }
    __syncthreads();

    // phase 2: M1-M3 for the tile + halo 1
    const T hdtdx = T(0.5) * dt * a.inv_dx, hdtdy = T(0.5) * dt * a.inv_dy;
    for (int k = tid; k < MPX * MPY; k += MTX * MTY) {
        const int px = k % MPX, py = k / MPX, rx = px + 1, ry = py + 1;
        const T z = s.raw[3][ry][rx];
        if (is_solid(z)) { s.wet[py][px] = 2; continue; }
        const T h = s.raw[0][ry][rx], qx = s.raw[1][ry][rx], qy = s.raw[2][ry][rx], eta = h + z;
        const bool wet = h > a.h_dry;
        s.wet[py][px] = wet ? 1 : 0;
        T sl[2][4];                                         // [x | y][eta, h, qx, qy]
#pragma unroll
        for (int d = 0; d < 2; ++d) {
            const int ax = rx - (d == 0), ay = ry - (d == 1), bx = rx + (d == 0), by = ry + (d == 1);
            const T za = s.raw[3][ay][ax], zb = s.raw[3][by][bx];
            const T ha = s.raw[0][ay][ax], hb = s.raw[0][by][bx];
            sl[d][0] = sl[d][1] = sl[d][2] = sl[d][3] = T(0);
            if (!is_solid(za) && !is_solid(zb) && wet && ha > a.h_dry && hb > a.h_dry) {
                sl[d][0] = minmod(eta - (ha + za), (hb + zb) - eta);
                sl[d][1] = minmod(h - ha, hb - h);
                sl[d][2] = minmod(qx - s.raw[1][ay][ax], s.raw[1][by][bx] - qx);
                sl[d][3] = minmod(qy - s.raw[2][ay][ax], s.raw[2][by][bx] - qy);
            }
        }
        T fe[4], fh[4], fqx[4], fqy[4];                    // M2: 0 W, 1 E, 2 S, 3 N
#pragma unroll
        for (int f = 0; f < 4; ++f) {
            const T sg = (f & 1) ? T(0.5) : T(-0.5);
            const T *q = sl[f >> 1];
            fe[f] = eta + sg * q[0]; fh[f] = h + sg * q[1]; fqx[f] = qx + sg * q[2]; fqy[f] = qy + sg * q[3];
        }
        // M3
        const T uE = face_vel(wet, fqx[1], fh[1], a.h_dry), uW = face_vel(wet, fqx[0], fh[0], a.h_dry);
        const T vN = face_vel(wet, fqy[3], fh[3], a.h_dry), vS = face_vel(wet, fqy[2], fh[2], a.h_dry);
        const T dh = -hdtdx * (fqx[1] - fqx[0]) - hdtdy * (fqy[3] - fqy[2]);
        const T dqx = -hdtdx * ((fqx[1] * uE - fqx[0] * uW) + a.g * T(0.5) * (fh[1] + fh[0]) * (fe[1] - fe[0]))
                      - hdtdy * (fqx[3] * vN - fqx[2] * vS);
        const T dqy = -hdtdx * (fqy[1] * uE - fqy[0] * uW)
                      - hdtdy * ((fqy[3] * vN - fqy[2] * vS) + a.g * T(0.5) * (fh[3] + fh[2]) * (fe[3] - fe[2]));
#pragma unroll
        for (int f = 0; f < 4; ++f) {
            const T hp = fmax(T(0), fh[f] + dh);
            const T r = wet ? fast_rcp(fmax(hp, a.h_dry)) : T(0);     // face velocity of a wet cell: q / max(h, h_dry); else 0
            s.fv[f][0][py][px] = hp;
            s.fv[f][1][py][px] = (fqx[f] + dqx) * r;
            s.fv[f][2][py][px] = (fqy[f] + dqy) * r;
            s.fv[f][3][py][px] = fe[f] - fh[f];
        }
    }
    __syncthreads();

    // phase 3a: M4, every face of the tile ONCE.  x-face fx of row py lies between predicted cells (fx, py) and
    // (fx + 1, py): the left one contributes its E face value, the right one its W face value; y-faces likewise
    // with N | S.  A solid / outside side is the wall ghost of the other (O2.1), or, on an open domain edge, its
    // transmissive ghost (D1).  Stored: mass flux, normal-momentum flux as seen by the left / lower and by the
    // right / upper cell (F1 - g h*^2/2 + g h_f^2/2 with h_f that cell's own face depth), tangential flux.
    constexpr int NXF = MTY * (MTX + 1), NYF = (MTY + 1) * MTX;
    for (int k = tid; k < NXF + NYF; k += MTX * MTY) {
        const bool xdir = k < NXF;
        const int kk = xdir ? k : k - NXF;
        const int fx = xdir ? kk % (MTX + 1) : kk % MTX, fy = xdir ? kk / (MTX + 1) : kk / MTX;
        const int pxL = xdir ? fx : fx + 1, pyL = xdir ? fy + 1 : fy;             // left / lower cell (predicted coordinates)
        const int pxR = xdir ? fx + 1 : fx + 1, pyR = xdir ? fy + 1 : fy + 1;
        const int fL = xdir ? 1 : 3, fR = xdir ? 0 : 2;                           // its E | N face, the other's W | S face
        const int wL = s.wet[pyL][pxL], wR = s.wet[pyR][pxR];
        T f0 = T(0), FL = T(0), FR = T(0), f2 = T(0);
        if (wL != 2 || wR != 2) {
            T hL = s.fv[fL][0][pyL][pxL], zL = s.fv[fL][3][pyL][pxL];
            T nL = s.fv[fL][xdir ? 1 : 2][pyL][pxL], tL = s.fv[fL][xdir ? 2 : 1][pyL][pxL];
            T hR = s.fv[fR][0][pyR][pxR], zR = s.fv[fR][3][pyR][pxR];
            T nR = s.fv[fR][xdir ? 1 : 2][pyR][pxR], tR = s.fv[fR][xdir ? 2 : 1][pyR][pxR];
            const int giR = x0 + pxR - 1, gjR = y0 + pyR - 1, giL = x0 + pxL - 1, gjL = y0 + pyL - 1;   // global cells
            bool open_out = false;
            if (wL == 2) {                              // the right / upper cell is real
                const bool edge = xdir ? giR == 0 : gjR == 0;
                const bool op = edge && open_face(a, xdir ? 0 : 2, giR, gjR);
                hL = hR; zL = zR; tL = tR; nL = op ? nR : -nR;
                if (op) open_out = true;
            } else if (wR == 2) {
                const bool edge = xdir ? giL == a.nx - 1 : gjL == a.ny - 1;
                const bool op = edge && open_face(a, xdir ? 1 : 3, giL, gjL);
                hR = hL; zR = zL; tR = tL; nR = op ? nL : -nL;
                if (op) open_out = true;
            }
            T f1L, f1R;
            face_flux(a.g, hL, nL, tL, zL, hR, nR, tR, zR, f0, f1L, f1R, f2);
            FL = f1L + T(0.5) * a.g * hL * hL; FR = f1R + T(0.5) * a.g * hR * hR;
            // volume through an open face (D1): counted by the tile that owns the real cell
            if (open_out) {
                const bool mine = wL == 2 ? (pxR >= 1 && pxR <= MTX && pyR >= 1 && pyR <= MTY) : (pxL >= 1 && pxL <= MTX && pyL >= 1 && pyL <= MTY);
                if (mine) add_outflow(a, dt, wL == 2 ? -f0 : f0, xdir ? a.inv_dx : a.inv_dy);
            }
        }
        T *dst = xdir ? &s.xf[0][fy][fx] : &s.yf[0][fy][fx];
        const int plane = xdir ? MTY * (MTX + 1) : (MTY + 1) * MTX;
        dst[0] = f0; dst[plane] = FL; dst[2 * plane] = FR; dst[3 * plane] = f2;
    }
    __syncthreads();

    // phase 3b: M5-M7 for my cell
    const int i = x0 + threadIdx.x, j = y0 + threadIdx.y;
    T lam = T(0);
    if (i < a.nx && j < a.ny) {
        const int c = j * a.nx + i, tx = threadIdx.x, ty = threadIdx.y, px = tx + 1, py = ty + 1;
        T hn = T(0), qxn = T(0), qyn = T(0);
        if (s.wet[py][px] != 2) {
            T FW0 = s.xf[0][ty][tx], FE0 = s.xf[0][ty][tx + 1], GS0 = s.yf[0][ty][tx], GN0 = s.yf[0][ty + 1][tx];
            const T FnW = s.xf[2][ty][tx], FnE = s.xf[1][ty][tx + 1], FtW = s.xf[3][ty][tx], FtE = s.xf[3][ty][tx + 1];
            const T GnS = s.yf[2][ty][tx], GnN = s.yf[1][ty + 1][tx], GtS = s.yf[3][ty][tx], GtN = s.yf[3][ty + 1][tx];
            if (i == 0) FW0 += qin * T(a.inflow[0][j]);
            if (i == a.nx - 1) FE0 -= qin * T(a.inflow[1][j]);
            if (j == 0) GS0 += qin * T(a.inflow[2][i]);
            if (j == a.ny - 1) GN0 -= qin * T(a.inflow[3][i]);
            // M5, folded into the flux differences: -dt/dx (dF - S dx)
            const T Sx = T(0.5) * a.g * (s.fv[0][0][py][px] + s.fv[1][0][py][px]) * (s.fv[0][3][py][px] - s.fv[1][3][py][px]);
            const T Sy = T(0.5) * a.g * (s.fv[2][0][py][px] + s.fv[3][0][py][px]) * (s.fv[2][3][py][px] - s.fv[3][3][py][px]);
            finish_cell(a, dt, s.raw[0][py + 1][px + 1], s.raw[1][py + 1][px + 1], s.raw[2][py + 1][px + 1],
                        FE0 - FW0, (FnE - FnW) - Sx, FtE - FtW,
                        GN0 - GS0, GtN - GtS, (GnN - GnS) - Sy,
                        a.n0[c], (int)OCC[c], hn, qxn, qyn, lam);
        }
        a.h[p ^ 1][c] = hn; a.qx[p ^ 1][c] = qxn; a.qy[p ^ 1][c] = qyn;
    }
    block_max_lambda(a.ctl, lam, s.red);
}

}  // namespace fp
