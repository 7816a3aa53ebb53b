// flood_march2.cuh -- variant 3 of step (F)+(T): the row-marching flood-cell update of
// flood_march.cuh (Eq. (2); same face flux face_eta(); branch-free finish_hat2()), with CPT
// adjacent columns per thread.
//
//   Why: ncu (profiles/r1_ncu_full_c5.md) shows variant 2 issue-bound (77 % of issue slots, about
//   285 instructions per cell, ~85 of them addressing, shared-memory exchange, loop and vote
//   overhead per thread-row).  With CPT = 2 a thread loads its cells with one 64-bit (fp32) or
//   128-bit (fp64) access per field, the face between its own cells never leaves registers, and
//   the per-thread-row overhead is spent once per CPT cells.
//
//   Geometry is that of variant 2 (strips of MW = 256 columns, chunks of R rows, the same
//   chunk_flag fast/general split); a CTA has MW / CPT threads.  Needs nx % CPT == 0.
#pragma once

#include "flood_march.cuh"

namespace fp {

template <int CPT> struct __align__(CPT) ByteN { uint8_t v[CPT]; };

template <typename T, int CPT>
struct March2Smem {
    static constexpr int NT = MW / CPT;
    T st[2][4][NT];                   // eta, u, v, z of each thread's LAST column, by row parity
    T fx[2][3][NT];                   // west-face flux (f0, f1L, f2) of each thread's FIRST column
    T er[3][MARCH_MAX_R];             // east-edge face of the strip for every row of the chunk
    T sw[4][MARCH_MAX_R];             // state of column x0-1 for every row of the chunk
    T red[32];
};

// finish_hat() of flood_march.cuh without divergent branches: the clamp (C12) is accumulated in
// registers (count, depth) and flushed once per chunk; friction (C6) and the wave speed
// are evaluated on max(h, h_dry) and selected.
template <typename T>
__device__ __forceinline__ void finish_hat2(const FloodArgs<T> &a, T dt, T &hn, T &qxn, T &qyn, T n0, int np,
                                            T &lam, T &clamp_h, int &clamp_n)
{
    const bool neg = hn < T(0);
    clamp_h += neg ? -hn : T(0);
    clamp_n += neg ? 1 : 0;
    hn = fmax(hn, T(0));
    const bool wet = hn > a.h_dry;
    const T hs = fmax(hn, a.h_dry);
    const T n = a.couple ? n0 * (T(1) + T(min(np, a.n_cap))) : n0;
    const T D = T(1) + dt * a.g * n * n * fast_sqrt(qxn * qxn + qyn * qyn) * pow_m73(hs);
    const T rD = wet ? fast_rcp(D) : T(0);
    qxn *= rD; qyn *= rD;
    const T rh = fast_rcp(hs), c = fast_sqrt(a.g * hs);
    const T l = fmax((fabs(qxn * rh) + c) * a.inv_dx, (fabs(qyn * rh) + c) * a.inv_dy);
    lam = fmax(lam, wet ? l : T(0));
}

template <typename T, int CPT> struct RawN { VecN<T, CPT> h, qx, qy, z; };

template <typename T, int CPT, bool GEN>
__device__ __forceinline__ RawN<T, CPT> march2_load(const T *__restrict__ H, const T *__restrict__ QX,
                                                    const T *__restrict__ QY, const T *__restrict__ Z,
                                                    int i, int j, int nx, int ny)
{
    RawN<T, CPT> r;
    if (GEN && (i >= nx || j < 0 || j >= ny)) {        // nx % CPT == 0: a thread is all in or all out
#pragma unroll
        for (int k = 0; k < CPT; ++k) { r.h.v[k] = r.qx.v[k] = r.qy.v[k] = T(0); r.z.v[k] = solid_z<T>(); }
        return r;
    }
    const size_t c = (size_t)j * nx + i;
    r.h = *reinterpret_cast<const VecN<T, CPT> *>(H + c);
    r.qx = *reinterpret_cast<const VecN<T, CPT> *>(QX + c);
    r.qy = *reinterpret_cast<const VecN<T, CPT> *>(QY + c);
    r.z = *reinterpret_cast<const VecN<T, CPT> *>(Z + c);
    return r;
}

template <typename T, int CPT, bool GEN>
__device__ __forceinline__ T march2_chunk(const FloodArgs<T> &a, March2Smem<T, CPT> &s, int x0, int y0, int R)
{
    constexpr int NT = MW / CPT;
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
    const int i = x0 + tid * CPT;                      // first of my columns
    const bool col_ok = GEN ? (i < nx) : true;
    const int y1 = min(y0 + R, ny);                    // rows [y0, y1) are owned by this chunk

    RawN<T, CPT> rp = march2_load<T, CPT, GEN>(H, QX, QY, Z, i, y0 - 1, nx, ny);
    RawN<T, CPT> c0 = march2_load<T, CPT, GEN>(H, QX, QY, Z, i, y0, nx, ny);
    RawN<T, CPT> c1 = march2_load<T, CPT, GEN>(H, QX, QY, Z, i, min(y0 + 1, GEN ? y0 + 1 : y1), nx, ny);

    // ---- pre-pass: strip-edge data for every row of the chunk (as in variant 2)
    for (int k = tid; k < R; k += NT) {                // east-edge face between columns x0+MW-1 and x0+MW
        const int j = y0 + k;
        T f0 = T(0), f1L = T(0), f1R, f2 = T(0);
        if (j < y1) {
            Raw4<T> l = march_load<T, GEN>(H, QX, QY, Z, x0 + MW - 1, j, nx, ny);
            Raw4<T> r = march_load<T, GEN>(H, QX, QY, Z, x0 + MW, j, nx, ny);
            T el, ul, vl, er_, ur, vr;
            march_prims<T, GEN>(l, h_dry, el, ul, vl);
            march_prims<T, GEN>(r, h_dry, er_, ur, vr);
            face_eta<T, GEN, false>(g, el, ul, vl, l.z, er_, ur, vr, r.z, f0, f1L, f1R, f2);
        }
        s.er[0][k] = f0; s.er[1][k] = f1L; s.er[2][k] = f2;
    }
    for (int k = tid; k < R; k += NT) {                // state of column x0-1
        Raw4<T> l = march_load<T, true>(H, QX, QY, Z, x0 - 1, min(y0 + k, ny - 1), nx, ny);
        T el, ul, vl;
        march_prims<T, true>(l, h_dry, el, ul, vl);
        s.sw[0][k] = el; s.sw[1][k] = ul; s.sw[2][k] = vl; s.sw[3][k] = l.z;
    }

    // halo row y0-1 becomes "prev"
    T eta_p[CPT], u_p[CPT], v_p[CPT], z_p[CPT];
#pragma unroll
    for (int k = 0; k < CPT; ++k) {
        Raw4<T> q{rp.h.v[k], rp.qx.v[k], rp.qy.v[k], rp.z.v[k]};
        march_prims<T, GEN>(q, h_dry, eta_p[k], u_p[k], v_p[k]);
        z_p[k] = q.z;
    }
    T ah[CPT], ax[CPT], ay[CPT], n0_p[CPT];            // accumulators of the previous (owned) row
    int occ_p[CPT];
#pragma unroll
    for (int k = 0; k < CPT; ++k) { ah[k] = ax[k] = ay[k] = n0_p[k] = T(0); occ_p[k] = 0; }
    T lam = T(0), clamp_h = T(0);
    int clamp_n = 0;

#pragma unroll 2
    for (int jj = y0; jj <= y1; ++jj) {
        RawN<T, CPT> cur = c0;
        c0 = c1;
        c1 = march2_load<T, CPT, GEN>(H, QX, QY, Z, i, GEN ? jj + 2 : min(jj + 2, y1), nx, ny);
        T eta[CPT], u[CPT], v[CPT], z[CPT], hc[CPT], qxc[CPT], qyc[CPT];
#pragma unroll
        for (int k = 0; k < CPT; ++k) {
            Raw4<T> q{cur.h.v[k], cur.qx.v[k], cur.qy.v[k], cur.z.v[k]};
            march_prims<T, GEN>(q, h_dry, eta[k], u[k], v[k]);
            z[k] = q.z; hc[k] = q.h; qxc[k] = q.qx; qyc[k] = q.qy;
        }
        const int b = jj & 1;
        s.st[b][0][tid] = eta[CPT - 1]; s.st[b][1][tid] = u[CPT - 1];
        s.st[b][2][tid] = v[CPT - 1];   s.st[b][3][tid] = z[CPT - 1];
        VecN<T, CPT> n0_c; ByteN<CPT> occ_c;
#pragma unroll
        for (int k = 0; k < CPT; ++k) { n0_c.v[k] = T(0); occ_c.v[k] = 0; }
        if (jj < y1 && col_ok) {
            const size_t c = (size_t)jj * nx + i;
            n0_c = *reinterpret_cast<const VecN<T, CPT> *>(a.n0 + c);
            if (a.couple) occ_c = *reinterpret_cast<const ByteN<CPT> *>(OCC + c);
        }
        __syncthreads();

        // south faces of the current row = north faces of the previous one (normal velocity v)
        T g0[CPT], g1L[CPT], g1R[CPT], g2[CPT];
#pragma unroll
        for (int k = 0; k < CPT; ++k)
            face_eta<T, GEN, true>(g, eta_p[k], v_p[k], u_p[k], z_p[k], eta[k], v[k], u[k], z[k], g0[k], g1L[k], g1R[k], g2[k]);

        if (jj > y0) {                                 // finish row jj-1
            const int j = jj - 1, bp = b ^ 1;
            const T *fe = (tid == NT - 1) ? &s.er[0][j - y0] : &s.fx[bp][0][tid + 1];
            const int stride = (tid == NT - 1) ? MARCH_MAX_R : NT;
            VecN<T, CPT> ho, qxo, qyo;
#pragma unroll
            for (int k = 0; k < CPT; ++k) {
                T hn = ah[k] - dtdy * g0[k], qxn = ax[k] - dtdy * g2[k], qyn = ay[k] - dtdy * g1L[k];
                if (k == CPT - 1) {                    // east face of my last column: from the right neighbour
                    hn -= dtdx * fe[0]; qxn -= dtdx * fe[stride]; qyn -= dtdx * fe[2 * stride];
                    if (GEN && i + k == nx - 1) hn += dtdx * qin * T(a.inflow[1][j]);
                }
                if (GEN && j == ny - 1 && col_ok) hn += dtdy * qin * T(a.inflow[3][i + k]);
                if (GEN && is_solid(z_p[k])) { hn = qxn = qyn = T(0); }
                else finish_hat2(a, dt, hn, qxn, qyn, n0_p[k], occ_p[k], lam, clamp_h, clamp_n);
                ho.v[k] = hn; qxo.v[k] = qxn; qyo.v[k] = qyn;
            }
            if (col_ok) {
                const size_t c = (size_t)j * nx + i;
                *reinterpret_cast<VecN<T, CPT> *>(Ho + c) = ho;
                *reinterpret_cast<VecN<T, CPT> *>(QXo + c) = qxo;
                *reinterpret_cast<VecN<T, CPT> *>(QYo + c) = qyo;
            }
        }
        if (jj < y1) {                                 // enter row jj: west faces, start its accumulators
            const T *sl = (tid == 0) ? &s.sw[0][jj - y0] : &s.st[b][0][tid - 1];
            const int stride = (tid == 0) ? MARCH_MAX_R : NT;
            T f0[CPT], f1L[CPT], f1R[CPT], f2[CPT];
            face_eta<T, GEN, true>(g, sl[0], sl[stride], sl[2 * stride], sl[3 * stride], eta[0], u[0], v[0], z[0],
                                   f0[0], f1L[0], f1R[0], f2[0]);
#pragma unroll
            for (int k = 1; k < CPT; ++k)
                face_eta<T, GEN, true>(g, eta[k - 1], u[k - 1], v[k - 1], z[k - 1], eta[k], u[k], v[k], z[k],
                                       f0[k], f1L[k], f1R[k], f2[k]);
            s.fx[b][0][tid] = f0[0]; s.fx[b][1][tid] = f1L[0]; s.fx[b][2][tid] = f2[0];
#pragma unroll
            for (int k = 0; k < CPT; ++k) {
                ah[k] = hc[k] + dtdx * f0[k] + dtdy * g0[k];
                ax[k] = qxc[k] + dtdx * f1R[k] + dtdy * g2[k];
                ay[k] = qyc[k] + dtdx * f2[k] + dtdy * g1R[k];
                if (k < CPT - 1) {                     // east face of column k = west face of column k+1
                    ah[k] -= dtdx * f0[k + 1]; ax[k] -= dtdx * f1L[k + 1]; ay[k] -= dtdx * f2[k + 1];
                }
                if (GEN && i + k == 0) ah[k] += dtdx * qin * T(a.inflow[0][jj]);
                if (GEN && jj == 0 && col_ok) ah[k] += dtdy * qin * T(a.inflow[2][i + k]);
            }
        }
#pragma unroll
        for (int k = 0; k < CPT; ++k) {
            eta_p[k] = eta[k]; u_p[k] = u[k]; v_p[k] = v[k]; z_p[k] = z[k];
            n0_p[k] = n0_c.v[k]; occ_p[k] = occ_c.v[k];
        }
    }
    if (clamp_n) {                                     // C12 accounting, once per thread and chunk
        atomicAdd(&a.ctl->clamped_volume, (double)clamp_h * (double)a.cell_area);
        atomicAdd(&a.ctl->neg_clamps, (unsigned long long)clamp_n);
    }
    return lam;
}

template <typename T, int CPT>
__global__ void __launch_bounds__(MW / CPT, sizeof(T) == 4 ? 4 : 2) flood_march2_kernel(FloodArgs<T> a)
{
    pdl_enter();
    constexpr int NT = MW / CPT;
    __shared__ March2Smem<T, CPT> s;
    if (a.ctl->halt) return;
    const int x0 = blockIdx.x * MW, y0 = blockIdx.y * a.R;
    const bool gen = a.chunk_flag[blockIdx.y * gridDim.x + blockIdx.x] != 0;
    T lam = gen ? march2_chunk<T, CPT, true>(a, s, x0, y0, a.R) : march2_chunk<T, CPT, false>(a, s, x0, y0, a.R);
    const int tid = threadIdx.x;
    for (int o = 16; o > 0; o >>= 1) lam = fmax(lam, __shfl_xor_sync(0xffffffffu, lam, o));
    __syncthreads();
    if ((tid & 31) == 0) s.red[tid >> 5] = lam;
    __syncthreads();
    if (tid < 32) {
        T m = tid < NT / 32 ? s.red[tid] : T(0);
        for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (tid == 0 && m > T(0)) atomic_max_lambda(a.ctl, (double)m);
    }
}

}  // namespace fp
