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
//   phase 3  every thread: the four faces of its cell (own face value | neighbour's opposite face
//            value, or the wall ghost), sources, finish_cell(), block-wide max of the wave speed.
// Algorithmic bytes per cell are those of the first-order step (33 B fp32); the halo-2 re-reads
// are L2 traffic.  Each face is evaluated by both of its cells (simple; ~2x the flux flops).
#pragma once

#include "flood.cuh"

namespace fp {

constexpr int MTX = 32, MTY = 8;                       // tile
constexpr int MRX = MTX + 4, MRY = MTY + 4;            // raw state: halo 2
constexpr int MPX = MTX + 2, MPY = MTY + 2;            // predicted face values: halo 1

template <typename T>
struct MusclSmem {
    T raw[4][MRY][MRX];            // h, qx, qy, z
    T fv[4][4][MPY][MPX];          // [face W,E,S,N][h, qx, qy, z]
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
            s.fv[f][0][py][px] = fmax(T(0), fh[f] + dh);
            s.fv[f][1][py][px] = fqx[f] + dqx;
            s.fv[f][2][py][px] = fqy[f] + dqy;
            s.fv[f][3][py][px] = fe[f] - fh[f];
        }
    }
    __syncthreads();

    // phase 3: M4-M7 for my cell
    const int i = x0 + threadIdx.x, j = y0 + threadIdx.y;
    T lam = T(0);
    if (i < a.nx && j < a.ny) {
        const int c = j * a.nx + i, px = threadIdx.x + 1, py = threadIdx.y + 1;
        T hn = T(0), qxn = T(0), qyn = T(0);
        if (s.wet[py][px] != 2) {
            const bool wet = s.wet[py][px] == 1;
            T F0[4], Fn[4], Ft[4], hf[4], zf[4];
            bool open[4];
#pragma unroll
            for (int f = 0; f < 4; ++f) {
                const int di = (f == 1) - (f == 0), dj = (f == 3) - (f == 2);
                const T hi = s.fv[f][0][py][px], zi = s.fv[f][3][py][px];
                const T ui = face_vel(wet, s.fv[f][1][py][px], hi, a.h_dry), vi = face_vel(wet, s.fv[f][2][py][px], hi, a.h_dry);
                const T uni = f < 2 ? ui : vi, uti = f < 2 ? vi : ui;
                T hk = hi, unk = -uni, utk = uti, zk = zi;                   // wall ghost (O2.1)
                const int wk = s.wet[py + dj][px + di];
                const bool edge = f == 0 ? i == 0 : f == 1 ? i == a.nx - 1 : f == 2 ? j == 0 : j == a.ny - 1;
                open[f] = edge && open_face(a, f, i, j);
                if (open[f]) unk = uni;                                      // transmissive ghost (D1)
                else if (wk != 2) {
                    const int g = f ^ 1;
                    hk = s.fv[g][0][py + dj][px + di]; zk = s.fv[g][3][py + dj][px + di];
                    const T uk = face_vel(wk == 1, s.fv[g][1][py + dj][px + di], hk, a.h_dry);
                    const T vk = face_vel(wk == 1, s.fv[g][2][py + dj][px + di], hk, a.h_dry);
                    unk = f < 2 ? uk : vk; utk = f < 2 ? vk : uk;
                }
                T f0, f1L, f1R, f2;
                if (f & 1) face_flux(a.g, hi, uni, uti, zi, hk, unk, utk, zk, f0, f1L, f1R, f2);
                else { face_flux(a.g, hk, unk, utk, zk, hi, uni, uti, zi, f0, f1R, f1L, f2); }   // f1L: as seen by my cell
                F0[f] = f0; Fn[f] = f1L + T(0.5) * a.g * hi * hi; Ft[f] = f2;
                hf[f] = hi; zf[f] = zi;
            }
            if (i == 0) F0[0] += qin * T(a.inflow[0][j]);
            if (i == a.nx - 1) F0[1] -= qin * T(a.inflow[1][j]);
            if (j == 0) F0[2] += qin * T(a.inflow[2][i]);
            if (j == a.ny - 1) F0[3] -= qin * T(a.inflow[3][i]);
            if (open[1]) add_outflow(a, dt, F0[1], a.inv_dx);
            if (open[0]) add_outflow(a, dt, -F0[0], a.inv_dx);
            if (open[3]) add_outflow(a, dt, F0[3], a.inv_dy);
            if (open[2]) add_outflow(a, dt, -F0[2], a.inv_dy);
            // M5, folded into the flux differences: -dt/dx (dF - S dx)
            const T Sx = T(0.5) * a.g * (hf[0] + hf[1]) * (zf[0] - zf[1]);
            const T Sy = T(0.5) * a.g * (hf[2] + hf[3]) * (zf[2] - zf[3]);
            finish_cell(a, dt, s.raw[0][py + 1][px + 1], s.raw[1][py + 1][px + 1], s.raw[2][py + 1][px + 1],
                        F0[1] - F0[0], (Fn[1] - Fn[0]) - Sx, Ft[1] - Ft[0],
                        F0[3] - F0[2], Ft[3] - Ft[2], (Fn[3] - Fn[2]) - Sy,
                        a.n0[c], (int)OCC[c], hn, qxn, qyn, lam);
        }
        a.h[p ^ 1][c] = hn; a.qx[p ^ 1][c] = qxn; a.qy[p ^ 1][c] = qyn;
    }
    block_max_lambda(a.ctl, lam, s.red);
}

}  // namespace fp
