// flood_wmarch.cuh -- variant 5 of step (F)+(T): the row-marching flood-cell update (Eq. (2),
// P:L105; face flux face_eta() of flood_march.cuh, finish_hat2() of flood_march2.cuh) with every
// WARP marching on its own: no block-wide barrier inside the row loop.
//
//   Why: ncu of variant 2 (profiles/r1_ncu_full_c5.md) shows the barrier as the largest stall
//   reason (one __syncthreads per row across 8 warps) and the kernel issue-bound.
//
//   A warp owns 32 columns (one per lane) of the CTA's 256-column strip and marches over the R rows
//   of the chunk.  Per row a lane evaluates its west face and its south face; the west neighbour's
//   state arrives by __shfl_up, the east face's flux by __shfl_down in the same iteration, so only
//   the north flux is deferred (it is next row's south flux, in registers).  Lane 0's west state
//   and lane 31's east flux for all R rows come from a per-warp pre-pass kept in shared memory
//   (8 values per row, read as two 128-bit broadcasts).  The warp-edge face is thus evaluated twice
//   (once by each warp) with the same inlined function on the same operands, hence identically.
#pragma once

#include "flood_march2.cuh"

namespace fp {

constexpr int WM_WARPS = MW / 32;
constexpr int WM_MAX_R = 64;          // rows per chunk the per-warp edge buffers hold (march_R <= 64)

template <typename T> struct __align__(sizeof(T) * 4) Quad { T a, b, c, d; };

template <typename T>
struct WMarchSmem {
    Quad<T> sw[WM_WARPS][WM_MAX_R];    // eta, u, v, z of column xw0-1, per row
    Quad<T> er[WM_WARPS][WM_MAX_R];    // f0, f1L, f2 of the face between columns xw0+31 and xw0+32
    T red[32];
};

template <typename T> __device__ __forceinline__ T shfl_up1(T v) { return __shfl_up_sync(0xffffffffu, v, 1); }
template <typename T> __device__ __forceinline__ T shfl_down1(T v) { return __shfl_down_sync(0xffffffffu, v, 1); }

template <typename T, bool GEN>
__device__ __forceinline__ T wmarch_chunk(const FloodArgs<T> &a, WMarchSmem<T> &s, int x0, int y0, int R)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nx = a.nx, ny = a.ny;
    const int p = a.ctl->parity;
    const T *__restrict__ H = a.h[p], *__restrict__ QX = a.qx[p], *__restrict__ QY = a.qy[p];
    const T *__restrict__ Z = a.zs;
    T *__restrict__ Ho = a.h[p ^ 1], *__restrict__ QXo = a.qx[p ^ 1], *__restrict__ QYo = a.qy[p ^ 1];
    const T dt = (T)a.ctl->dt;
    const T qin = GEN ? (T)a.ctl->q_in : T(0);
    const T dtdx = dt * a.inv_dx, dtdy = dt * a.inv_dy;
    const T g = a.g, h_dry = a.h_dry;
    const int xw0 = x0 + warp * 32;
    const int i = xw0 + lane;
    const bool col_ok = GEN ? (i < nx) : true;
    const int y1 = min(y0 + R, ny);                    // rows [y0, y1) are owned by this chunk
    if (GEN && xw0 >= nx) return T(0);                 // whole warp outside the grid (warp-uniform)

    Raw4<T> rp = march_load<T, GEN>(H, QX, QY, Z, i, y0 - 1, nx, ny);
    Raw4<T> c0 = march_load<T, GEN>(H, QX, QY, Z, i, y0, nx, ny);
    Raw4<T> c1 = march_load<T, GEN>(H, QX, QY, Z, i, min(y0 + 1, GEN ? y0 + 1 : y1), nx, ny);

    // ---- pre-pass: warp-edge data for every row of the chunk
    Quad<T> *sw = s.sw[warp], *er = s.er[warp];
    for (int k = lane; k < R; k += 32) {
        const int j = min(y0 + k, ny - 1);
        Raw4<T> w = march_load<T, true>(H, QX, QY, Z, xw0 - 1, j, nx, ny);
        Raw4<T> l = march_load<T, GEN>(H, QX, QY, Z, xw0 + 31, j, nx, ny);
        Raw4<T> r = march_load<T, true>(H, QX, QY, Z, xw0 + 32, j, nx, ny);
        T ew, uw, vw, el, ul, vl, er_, ur, vr, f0, f1L, f1R, f2;
        march_prims<T, true>(w, h_dry, ew, uw, vw);
        march_prims<T, GEN>(l, h_dry, el, ul, vl);
        march_prims<T, true>(r, h_dry, er_, ur, vr);
        face_eta<T, true, false>(g, el, ul, vl, l.z, er_, ur, vr, r.z, f0, f1L, f1R, f2);
        sw[k] = Quad<T>{ew, uw, vw, w.z};
        er[k] = Quad<T>{f0, f1L, f2, T(0)};
    }
    __syncwarp();

    // halo row y0-1 becomes "prev"
    T eta_p, u_p, v_p, z_p;
    march_prims<T, GEN>(rp, h_dry, eta_p, u_p, v_p);
    z_p = rp.z;
    T ah = T(0), ax = T(0), ay = T(0), n0_p = T(0);    // accumulators of the previous (owned) row
    int occ_p = 0;
    T lam = T(0), clamp_h = T(0);
    int clamp_n = 0;

#pragma unroll 2
    for (int jj = y0; jj <= y1; ++jj) {
        Raw4<T> cur = c0;
        c0 = c1;
        c1 = march_load<T, GEN>(H, QX, QY, Z, i, GEN ? jj + 2 : min(jj + 2, y1), nx, ny);
        T eta, u, v;
        march_prims<T, GEN>(cur, h_dry, eta, u, v);
        T n0_c = T(0); int occ_c = 0;
        if (jj < y1 && col_ok) {
            const size_t c = (size_t)jj * nx + i;
            n0_c = a.n0[c];
            occ_c = a.couple ? (int)a.occ[c] : 0;
        }

        // south face of the current row = north face of the previous one (normal velocity v)
        T g0, g1L, g1R, g2;
        face_eta<T, GEN, true>(g, eta_p, v_p, u_p, z_p, eta, v, u, cur.z, g0, g1L, g1R, g2);

        if (jj > y0) {                                 // finish row jj-1
            const int j = jj - 1;
            T hn = ah - dtdy * g0, qxn = ax - dtdy * g2, qyn = ay - dtdy * g1L;
            if (GEN && j == ny - 1 && col_ok) hn += dtdy * qin * T(a.inflow[3][i]);
            if (GEN && is_solid(z_p)) { hn = qxn = qyn = T(0); }
            else finish_hat2(a, dt, hn, qxn, qyn, n0_p, occ_p, lam, clamp_h, clamp_n);
            if (col_ok) {
                const size_t c = (size_t)j * nx + i;
                Ho[c] = hn; QXo[c] = qxn; QYo[c] = qyn;
            }
        }
        if (jj < y1) {                                 // enter row jj: west and east faces, accumulators
            const int k = jj - y0;
            const Quad<T> ws = sw[k], ef = er[k];      // same address for all lanes: broadcast
            T el = shfl_up1(eta), ul = shfl_up1(u), vl = shfl_up1(v), zl = shfl_up1(cur.z);
            if (lane == 0) { el = ws.a; ul = ws.b; vl = ws.c; zl = ws.d; }
            T f0, f1L, f1R, f2;
            face_eta<T, GEN, true>(g, el, ul, vl, zl, eta, u, v, cur.z, f0, f1L, f1R, f2);
            T e0 = shfl_down1(f0), e1 = shfl_down1(f1L), e2 = shfl_down1(f2);
            if (lane == 31) { e0 = ef.a; e1 = ef.b; e2 = ef.c; }
            ah = cur.h + dtdx * (f0 - e0) + dtdy * g0;
            ax = cur.qx + dtdx * (f1R - e1) + dtdy * g2;
            ay = cur.qy + dtdx * (f2 - e2) + dtdy * g1R;
            if (GEN) {
                if (i == 0) ah += dtdx * qin * T(a.inflow[0][jj]);
                if (i == nx - 1) ah += dtdx * qin * T(a.inflow[1][jj]);
                if (jj == 0 && col_ok) ah += dtdy * qin * T(a.inflow[2][i]);
            }
        }
        eta_p = eta; u_p = u; v_p = v; z_p = cur.z; n0_p = n0_c; occ_p = occ_c;
    }
    if (clamp_n) {                                     // C12 accounting, once per thread and chunk
        atomicAdd(&a.ctl->clamped_volume, (double)clamp_h * (double)a.cell_area);
        atomicAdd(&a.ctl->neg_clamps, (unsigned long long)clamp_n);
    }
    return lam;
}

template <typename T>
__global__ void __launch_bounds__(MW, sizeof(T) == 4 ? 4 : 2) flood_wmarch_kernel(FloodArgs<T> a)
{
    __shared__ WMarchSmem<T> s;
    if (a.ctl->halt) return;
    const int x0 = blockIdx.x * MW, y0 = blockIdx.y * a.R;
    const bool gen = a.chunk_flag[blockIdx.y * gridDim.x + blockIdx.x] != 0;
    T lam = gen ? wmarch_chunk<T, true>(a, s, x0, y0, a.R) : wmarch_chunk<T, false>(a, s, x0, y0, a.R);
    const int tid = threadIdx.x;
    for (int o = 16; o > 0; o >>= 1) lam = fmax(lam, __shfl_xor_sync(0xffffffffu, lam, o));
    if ((tid & 31) == 0) s.red[tid >> 5] = lam;
    __syncthreads();
    if (tid < 32) {
        T m = tid < WM_WARPS ? s.red[tid] : T(0);
        for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (tid == 0 && m > T(0)) atomic_max_lambda(a.ctl, (double)m);
    }
}

}  // namespace fp
