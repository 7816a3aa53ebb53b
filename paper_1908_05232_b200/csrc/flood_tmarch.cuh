// flood_tmarch.cuh -- variant 4 of step (F)+(T): the row-marching flood-cell update of
// flood_march2.cuh (Eq. (2); same face flux, finish, strip/chunk geometry and shared-memory
// exchange) with the rows of an interior chunk brought in by the TMA engine and, in fp32, the
// arithmetic on packed pairs (flood_pk.cuh).  The default kernel from 2^22 cells.
//
//   Why TMA: ncu of variant 3 (two columns per thread, 117 registers, 16 warps/SM) showed the fewest
//   instructions per cell of the register-prefetch variants (195) but IPC 0.52 with long-scoreboard
//   (global-load latency) as the dominant stall: prefetching two rows ahead into registers does not
//   keep enough bytes in flight at that occupancy.  Here one elected lane of warp 0 issues, per row,
//   six 1-D bulk copies (cp.async.bulk global -> shared: h, qx, qy, z, n0 of the strip's 256 columns
//   and their N_p bytes) into a ring of STAGES row buffers, each completing on an mbarrier; the ring
//   runs STAGES rows ahead of the arithmetic at no register cost.  The slot read in iteration r is
//   refilled with row r+STAGES right after that iteration's barrier (every thread has its values in
//   registers by then).
//
//   chunk_flag picks the path of a chunk: 0 = interior without solid cells (no selects), 2 = interior
//   with solid cells in it or its halo (same path with wall-ghost selects, SOLID = true), 3 = touching
//   the domain edge with the strip inside the domain (EDGE = true: ghost rows of solid cells beyond the
//   edge, inflow faces, a short last chunk), 1 = edge chunk of a strip that sticks out of the domain
//   (march2_chunk<GEN=true>: plain loads, bounds checks, inflow).
//   Needs nx % 16 == 0 (16-byte alignment of every row segment).
//
//   TM_SPLIT_BARRIER=1 builds the measured-and-dropped alternative to the per-row __syncthreads: a
//   split-phase mbarrier (arrive after publishing, wait after the south faces), whose try_wait loop
//   spins through more issue slots than the barrier stall it removes.
#pragma once

#include <type_traits>

#include "flood_march2.cuh"
#include "flood_pk.cuh"

namespace fp {

#ifndef TM_SPLIT_BARRIER
#define TM_SPLIT_BARRIER 0
#endif

template <typename T>
struct __align__(16) RowStage {
    T h[MW], qx[MW], qy[MW], z[MW], n0[MW];
    uint8_t occ[MW];
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    // try_wait suspends the thread in hardware until the phase completes or the time hint (ns)
    // runs out; without the hint it returns after a short system-dependent time and the loop
    // spins through issue slots (ncu: 16 rounds per row on the exchange barrier)
    uint32_t ok;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n selp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity), "r"(100000u) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool elect_one()
{
    uint32_t ok;
    asm volatile("{\n .reg .pred p;\n elect.sync _|p, 0xffffffff;\n selp.u32 %0, 1, 0, p;\n}\n" : "=r"(ok));
    return ok != 0;
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// one row segment (columns x0 .. x0+MW-1 of row j) -> stage; EDGE: a row beyond the domain is the
// ghost row of solid cells (the wall, C13)
template <typename T, bool EDGE>
__device__ __forceinline__ void tm_issue_row(const FloodArgs<T> &a, const T *H, const T *QX, const T *QY, const uint8_t *OCC,
                                             RowStage<T> &st, uint64_t *bar, int x0, int j)
{
    constexpr uint32_t RB = MW * sizeof(T);
    mbar_expect_tx(bar, 5 * RB + MW);
    if (EDGE && (j < 0 || j >= a.ny)) {
        const int sd = j < 0 ? 0 : 1, p = H == a.h[1] ? 1 : 0;
        if (a.halo_z[sd]) {                            // row slab (8f-4): the neighbour slab's boundary row, read in place
            bulk_g2s(st.h, a.halo_h[sd][p] + x0, RB, bar);
            bulk_g2s(st.qx, a.halo_qx[sd][p] + x0, RB, bar);
            bulk_g2s(st.qy, a.halo_qy[sd][p] + x0, RB, bar);
            bulk_g2s(st.z, a.halo_z[sd] + x0, RB, bar);
            bulk_g2s(st.n0, a.ghost_zero, RB, bar);
            bulk_g2s(st.occ, a.ghost_occ, MW, bar);
            return;
        }
        bulk_g2s(st.h, a.ghost_zero, RB, bar);
        bulk_g2s(st.qx, a.ghost_zero, RB, bar);
        bulk_g2s(st.qy, a.ghost_zero, RB, bar);
        bulk_g2s(st.z, a.ghost_inf, RB, bar);
        bulk_g2s(st.n0, a.ghost_zero, RB, bar);
        bulk_g2s(st.occ, a.ghost_occ, MW, bar);
        return;
    }
    const size_t c = (size_t)j * a.nx + x0;
    bulk_g2s(st.h, H + c, RB, bar);
    bulk_g2s(st.qx, QX + c, RB, bar);
    bulk_g2s(st.qy, QY + c, RB, bar);
    bulk_g2s(st.z, a.zs + c, RB, bar);
    bulk_g2s(st.n0, a.n0 + c, RB, bar);
    bulk_g2s(st.occ, OCC + c, MW, bar);
}

// one chunk.  SOLID: solid cells in it or in its halo (wall-ghost selects).  EDGE (implies SOLID): it
// touches the domain edge: rows and columns beyond it are ghost solid cells, inflow faces add their
// discharge (C14), the last chunk of a strip may be shorter than R.
//
//   Synchronisation per row: the neighbour exchange (last-column state st[b], west-face flux
//   fx[b]) needs one CTA-wide barrier per row.  It sits AFTER the south faces, which need nothing
//   from the neighbours, so the skew between warps is spent on useful work first.  The ring slot is
//   refilled after that barrier (all threads have their values in registers by then).  The TMA issue sits in a warp-uniform branch with one elected
//   lane, its addresses derived from uniform values only.
template <typename T, int CPT, int STAGES, bool SOLID, bool EDGE>
__device__ __forceinline__ T tmarch_chunk(const FloodArgs<T> &a, March2Smem<T, CPT> &s, RowStage<T> *ring,
                                          uint64_t *bars, int x0, int y0, int Rfull, uint8_t *dry_out)
{
    const int R = EDGE ? min(Rfull, a.ny - y0) : Rfull;   // rows of this chunk inside the domain
    const T qin = EDGE ? (T)a.ctl->q_in : T(0);
    const int ny = a.ny;
    constexpr int NT = MW / CPT;
    const int tid = threadIdx.x;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);       // warp-uniform by construction
    const int nx = a.nx;
    const int p = __shfl_sync(0xffffffffu, a.ctl->parity, 0);
    const uint8_t *__restrict__ OCC = a.occ + (size_t)p * a.occ_stride;
    const T *__restrict__ H = a.h[p], *__restrict__ QX = a.qx[p], *__restrict__ QY = a.qy[p];
    const T *__restrict__ Z = a.zs;
    T *__restrict__ Ho = a.h[p ^ 1], *__restrict__ QXo = a.qx[p ^ 1], *__restrict__ QYo = a.qy[p ^ 1];
    const T dt = (T)a.ctl->dt;
    const T dtdx = dt * a.inv_dx, dtdy = dt * a.inv_dy;
    const T g = a.g, h_dry = a.h_dry;
    const int i = x0 + tid * CPT;
    const int nrows = R + 2;                           // ring row r holds grid row y0 - 1 + r
    uint64_t *xbar = bars + STAGES;                    // exchange barriers, by row parity

    if (tid == 0) {
        for (int k = 0; k < STAGES; ++k) mbar_init(&bars[k], 1);
        mbar_init(&xbar[0], NT); mbar_init(&xbar[1], NT);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (warp == 0) {
        if (elect_one())
            for (int r = 0; r < STAGES && r < nrows; ++r) tm_issue_row<T, EDGE>(a, H, QX, QY, OCC, ring[r], &bars[r], x0, y0 - 1 + r);
    }

    // ---- pre-pass: strip-edge data for every row of the chunk (as in variants 2, 3)
    for (int k = tid; k < R; k += NT) {
        const int j = y0 + k;
        Raw4<T> l = march_load<T, EDGE>(H, QX, QY, Z, x0 + MW - 1, j, nx, a.ny);
        Raw4<T> r = march_load<T, EDGE>(H, QX, QY, Z, x0 + MW, j, nx, a.ny);
        Raw4<T> w = march_load<T, EDGE>(H, QX, QY, Z, x0 - 1, j, nx, a.ny);
        T el, ul, vl, er_, ur, vr, ew, uw, vw, f0, f1L, f1R, f2;
        march_prims<T, SOLID>(l, h_dry, el, ul, vl);
        march_prims<T, SOLID>(r, h_dry, er_, ur, vr);
        march_prims<T, SOLID>(w, h_dry, ew, uw, vw);
        face_eta<T, SOLID, false>(g, el, ul, vl, l.z, er_, ur, vr, r.z, f0, f1L, f1R, f2);
        s.er[0][k] = f0; s.er[1][k] = f1L; s.er[2][k] = f2;
        s.sw[0][k] = ew; s.sw[1][k] = uw; s.sw[2][k] = vw; s.sw[3][k] = w.z;
    }

    // halo row y0-1 (ring row 0) becomes "prev"
    T eta_p[CPT], u_p[CPT], v_p[CPT], z_p[CPT];
    {
        mbar_wait(&bars[0], 0);
        const RowStage<T> &st = ring[0];
        const VecN<T, CPT> h = *reinterpret_cast<const VecN<T, CPT> *>(&st.h[tid * CPT]);
        const VecN<T, CPT> qx = *reinterpret_cast<const VecN<T, CPT> *>(&st.qx[tid * CPT]);
        const VecN<T, CPT> qy = *reinterpret_cast<const VecN<T, CPT> *>(&st.qy[tid * CPT]);
        const VecN<T, CPT> z = *reinterpret_cast<const VecN<T, CPT> *>(&st.z[tid * CPT]);
#pragma unroll
        for (int k = 0; k < CPT; ++k) {
            Raw4<T> q{h.v[k], qx.v[k], qy.v[k], z.v[k]};
            march_prims<T, SOLID>(q, h_dry, eta_p[k], u_p[k], v_p[k]);
            z_p[k] = q.z;
        }
    }
    __syncthreads();                                   // slot 0 consumed; er/sw visible
    if (warp == 0 && STAGES < nrows) {
        if (elect_one()) tm_issue_row<T, EDGE>(a, H, QX, QY, OCC, ring[0], &bars[0], x0, y0 - 1 + STAGES);
    }

    T ah[CPT], ax[CPT], ay[CPT], n0_p[CPT];
    int occ_p[CPT];
#pragma unroll
    for (int k = 0; k < CPT; ++k) { ah[k] = ax[k] = ay[k] = n0_p[k] = T(0); occ_p[k] = 0; }
    T lam = T(0), clamp_h = T(0);
    int clamp_n = 0;
    bool live_p = true;                                // anything but exact zeros in the accumulators?
    bool seg_live = false;                             // has my warp written anything but zeros in this chunk? (warp-uniform)

    // my addresses: the ring slot is followed by a running pointer (wraps after STAGES rows), the
    // exchange rows and barriers by compile-time offsets (the row loop is unrolled by two)
    const char *sp = reinterpret_cast<const char *>(ring) + sizeof(RowStage<T>) + tid * CPT * sizeof(T);   // slot 1
    const char *op = reinterpret_cast<const char *>(&ring[1].occ[tid * CPT]);
    uint64_t *tbar = &bars[1];
    int slot = 1;
    uint32_t tma_par = 0, xpar = 0;
    T *my_st = &s.st[0][0][tid];
    T *my_fx = &s.fx[0][0][tid];
    constexpr int ST_B = 4 * NT, FX_B = 3 * NT;         // stride of the row-parity index of st / fx
    const bool last_thread = tid == NT - 1, first_thread = tid == 0;
    T *out_h = Ho + (size_t)y0 * nx + i, *out_qx = QXo + (size_t)y0 * nx + i, *out_qy = QYo + (size_t)y0 * nx + i;
    const int nit = R + 1;                             // iteration it handles grid row y0 + it (ring row it + 1)

    if constexpr (std::is_same<T, float>::value && CPT % 2 == 0) {
    // ---- fp32: the columns of a thread as NP packed pairs (flood_pk.cuh)
    constexpr int NP = CPT / 2;
    f2 eta_q[NP], u_q[NP], v_q[NP], z_q[NP], ah2[NP], ax2[NP], ay2[NP], n0_q[NP];
    int occ_q[CPT];
#pragma unroll
    for (int k = 0; k < NP; ++k) {
        eta_q[k] = pk(eta_p[2 * k], eta_p[2 * k + 1]); u_q[k] = pk(u_p[2 * k], u_p[2 * k + 1]);
        v_q[k] = pk(v_p[2 * k], v_p[2 * k + 1]); z_q[k] = pk(z_p[2 * k], z_p[2 * k + 1]);
        ah2[k] = ax2[k] = ay2[k] = n0_q[k] = pk1(0.f);
        occ_q[2 * k] = occ_q[2 * k + 1] = 0;
    }
    const f2 dtdx2 = pk1(dtdx), dtdy2 = pk1(dtdy), ndtdy2 = pk1(-dtdy), ndtdx2 = pk1(-dtdx);

    auto row = [&](auto qc, int it) {
        constexpr int b = decltype(qc)::value;
        mbar_wait(tbar, tma_par);
        const RowStage<float> &st = *reinterpret_cast<const RowStage<float> *>(sp);
        VecN<f2, NP> hc = *reinterpret_cast<const VecN<f2, NP> *>(st.h), qxc = *reinterpret_cast<const VecN<f2, NP> *>(st.qx);
        VecN<f2, NP> qyc = *reinterpret_cast<const VecN<f2, NP> *>(st.qy);
        const VecN<f2, NP> z = *reinterpret_cast<const VecN<f2, NP> *>(st.z);
        const VecN<f2, NP> n0_c = *reinterpret_cast<const VecN<f2, NP> *>(st.n0);
        const ByteN<CPT> occ_c = *reinterpret_cast<const ByteN<CPT> *>(op);
        f2 eta[NP], u[NP], v[NP];
#pragma unroll
        for (int k = 0; k < NP; ++k) prims_x2<SOLID>(hc.v[k], qxc.v[k], qyc.v[k], z.v[k], h_dry, eta[k], u[k], v[k]);
        float *stb = my_st + b * ST_B;
        stb[0] = eta[NP - 1].y; stb[NT] = u[NP - 1].y; stb[2 * NT] = v[NP - 1].y; stb[3 * NT] = z.v[NP - 1].y;
#if TM_SPLIT_BARRIER
        mbar_arrive(&xbar[b]);                         // publishes st[b] of this row and fx[b^1] of the previous one
#endif

        // south faces of the current row = north faces of the previous one (normal velocity v)
        f2 g0[NP], g1L[NP], g1R[NP], g2[NP];
#pragma unroll
        for (int k = 0; k < NP; ++k)
            face_eta_x2<SOLID>(g, eta_q[k], v_q[k], u_q[k], z_q[k], eta[k], v[k], u[k], z.v[k], g0[k], g1L[k], g1R[k], g2[k]);

#if TM_SPLIT_BARRIER
        mbar_wait(&xbar[b], xpar);                     // use it/2 of xbar[b]
#else
        __syncthreads();                               // st[b] of this row and fx[b^1] of the previous one are visible
#endif
        if (warp == 0 && it + 1 + STAGES < nrows) {
            if (elect_one()) tm_issue_row<T, EDGE>(a, H, QX, QY, OCC, ring[slot], tbar, x0, y0 + it + STAGES);
        }
        sp += sizeof(RowStage<float>); op += sizeof(RowStage<float>); tbar += 1;
        if (++slot == STAGES) {
            slot = 0; tma_par ^= 1u;
            sp -= STAGES * sizeof(RowStage<float>); op -= STAGES * sizeof(RowStage<float>); tbar -= STAGES;
        }

        if (it > 0) {                                  // finish row y0 + it - 1
            const float *fe = last_thread ? &s.er[0][it - 1] : my_fx + (b ^ 1) * FX_B + 1;
            const int stride = last_thread ? MARCH_MAX_R : NT;
            const float e0 = fe[0], e1 = fe[stride], e2 = fe[2 * stride];
            // a warp whose cells of this row hold exact zeros and receive no flux writes zeros
            // (sign bits shifted out: -0 counts as zero)
            unsigned bits = __float_as_uint(e0) | __float_as_uint(e1) | __float_as_uint(e2);
#pragma unroll
            for (int k = 0; k < NP; ++k)
                bits |= __float_as_uint(g0[k].x) | __float_as_uint(g0[k].y) | __float_as_uint(g1L[k].x) | __float_as_uint(g1L[k].y)
                      | __float_as_uint(g2[k].x) | __float_as_uint(g2[k].y);
            const int jrow = y0 + it - 1;
            const bool live = live_p || (bits << 1) != 0u || (EDGE && (jrow == ny - 1 || i + CPT == nx));
            VecN<f2, NP> ho, qxo, qyo;
#pragma unroll
            for (int k = 0; k < NP; ++k) ho.v[k] = qxo.v[k] = qyo.v[k] = pk1(0.f);
            if (__any_sync(0xffffffffu, live)) {
                seg_live = true;
#pragma unroll
                for (int k = 0; k < NP; ++k) {
                    ho.v[k] = fma2(ndtdy2, g0[k], ah2[k]); qxo.v[k] = fma2(ndtdy2, g2[k], ax2[k]); qyo.v[k] = fma2(ndtdy2, g1L[k], ay2[k]);
                }
                ho.v[NP - 1].y = fmaf(-dtdx, e0, ho.v[NP - 1].y); qxo.v[NP - 1].y = fmaf(-dtdx, e1, qxo.v[NP - 1].y);
                qyo.v[NP - 1].y = fmaf(-dtdx, e2, qyo.v[NP - 1].y);
                if (EDGE) {                            // inflow faces on the east / north edge (C14)
                    if (i + CPT == nx) ho.v[NP - 1].y += dtdx * qin * float(a.inflow[1][jrow]);
                    if (jrow == ny - 1) {
#pragma unroll
                        for (int k = 0; k < NP; ++k) {
                            ho.v[k].x += dtdy * qin * float(a.inflow[3][i + 2 * k]);
                            ho.v[k].y += dtdy * qin * float(a.inflow[3][i + 2 * k + 1]);
                        }
                    }
                }
                if (SOLID) {                           // nothing moves in a solid cell (and no clamp is counted)
#pragma unroll
                    for (int k = 0; k < NP; ++k) {
                        if (is_solid(z_q[k].x)) { ho.v[k].x = qxo.v[k].x = qyo.v[k].x = 0.f; }
                        if (is_solid(z_q[k].y)) { ho.v[k].y = qxo.v[k].y = qyo.v[k].y = 0.f; }
                    }
                }
#pragma unroll
                for (int k = 0; k < NP; ++k)
                    finish_hat_x2(a, dt, ho.v[k], qxo.v[k], qyo.v[k], n0_q[k], occ_q[2 * k], occ_q[2 * k + 1], lam, clamp_h, clamp_n);
            }
            *reinterpret_cast<VecN<f2, NP> *>(out_h) = ho;
            *reinterpret_cast<VecN<f2, NP> *>(out_qx) = qxo;
            *reinterpret_cast<VecN<f2, NP> *>(out_qy) = qyo;
            out_h += nx; out_qx += nx; out_qy += nx;
        }
        if (it < R) {                                  // enter row y0 + it: west faces, start its accumulators
            const float *sl = first_thread ? &s.sw[0][it] : stb - 1;
            const int stride = first_thread ? MARCH_MAX_R : NT;
            // pair k: face .x = (column 2k-1 | column 2k), face .y = (column 2k | column 2k+1)
            f2 f0[NP], f1L[NP], f1R[NP], f2v[NP];
#pragma unroll
            for (int k = 0; k < NP; ++k) {
                const f2 le = k == 0 ? pk(sl[0], eta[0].x) : pk(eta[k - 1].y, eta[k].x);
                const f2 lu = k == 0 ? pk(sl[stride], u[0].x) : pk(u[k - 1].y, u[k].x);
                const f2 lv = k == 0 ? pk(sl[2 * stride], v[0].x) : pk(v[k - 1].y, v[k].x);
                const f2 lz = k == 0 ? pk(sl[3 * stride], z.v[0].x) : pk(z.v[k - 1].y, z.v[k].x);
                face_eta_x2<SOLID>(g, le, lu, lv, lz, eta[k], u[k], v[k], z.v[k], f0[k], f1L[k], f1R[k], f2v[k]);
            }
            float *fxb = my_fx + b * FX_B;
            fxb[0] = f0[0].x; fxb[NT] = f1L[0].x; fxb[2 * NT] = f2v[0].x;
            unsigned ab = 0u;
#pragma unroll
            for (int k = 0; k < NP; ++k) {
                ah2[k] = fma2(dtdx2, f0[k], fma2(dtdy2, g0[k], hc.v[k]));
                ax2[k] = fma2(dtdx2, f1R[k], fma2(dtdy2, g2[k], qxc.v[k]));
                ay2[k] = fma2(dtdx2, f2v[k], fma2(dtdy2, g1R[k], qyc.v[k]));
                if (k < NP - 1) {                      // east faces of both columns: the next west faces
                    ah2[k] = fma2(ndtdx2, pk(f0[k].y, f0[k + 1].x), ah2[k]);
                    ax2[k] = fma2(ndtdx2, pk(f1L[k].y, f1L[k + 1].x), ax2[k]);
                    ay2[k] = fma2(ndtdx2, pk(f2v[k].y, f2v[k + 1].x), ay2[k]);
                } else {                               // east face of the first column; the second one's comes from the neighbour
                    ah2[k].x = fmaf(-dtdx, f0[k].y, ah2[k].x); ax2[k].x = fmaf(-dtdx, f1L[k].y, ax2[k].x);
                    ay2[k].x = fmaf(-dtdx, f2v[k].y, ay2[k].x);
                }
                if (EDGE) {                            // inflow faces on the west / south edge (C14)
                    if (k == 0 && i == 0) ah2[0].x += dtdx * qin * float(a.inflow[0][y0 + it]);
                    if (y0 + it == 0) {
                        ah2[k].x += dtdy * qin * float(a.inflow[2][i + 2 * k]);
                        ah2[k].y += dtdy * qin * float(a.inflow[2][i + 2 * k + 1]);
                    }
                }
                ab |= __float_as_uint(ah2[k].x) | __float_as_uint(ah2[k].y) | __float_as_uint(ax2[k].x)
                    | __float_as_uint(ax2[k].y) | __float_as_uint(ay2[k].x) | __float_as_uint(ay2[k].y);
            }
            live_p = (ab << 1) != 0u;
        }
#pragma unroll
        for (int k = 0; k < NP; ++k) {
            eta_q[k] = eta[k]; u_q[k] = u[k]; v_q[k] = v[k]; z_q[k] = z.v[k];
            n0_q[k] = n0_c.v[k];
            occ_q[2 * k] = a.couple ? (int)occ_c.v[2 * k] : 0; occ_q[2 * k + 1] = a.couple ? (int)occ_c.v[2 * k + 1] : 0;
        }
    };

    for (int base = 0; base < nit; base += 2) {
        row(std::integral_constant<int, 0>{}, base);
        if (base + 1 < nit) row(std::integral_constant<int, 1>{}, base + 1);
        xpar ^= 1u;
    }
    } else {
    auto row = [&](auto qc, int it) {
        constexpr int b = decltype(qc)::value;
        mbar_wait(tbar, tma_par);
        const RowStage<T> &st = *reinterpret_cast<const RowStage<T> *>(sp);
        const VecN<T, CPT> hv = *reinterpret_cast<const VecN<T, CPT> *>(st.h);
        const VecN<T, CPT> qxv = *reinterpret_cast<const VecN<T, CPT> *>(st.qx);
        const VecN<T, CPT> qyv = *reinterpret_cast<const VecN<T, CPT> *>(st.qy);
        const VecN<T, CPT> zv = *reinterpret_cast<const VecN<T, CPT> *>(st.z);
        const VecN<T, CPT> n0_c = *reinterpret_cast<const VecN<T, CPT> *>(st.n0);
        const ByteN<CPT> occ_c = *reinterpret_cast<const ByteN<CPT> *>(op);
        T eta[CPT], u[CPT], v[CPT], z[CPT], hc[CPT], qxc[CPT], qyc[CPT];
#pragma unroll
        for (int k = 0; k < CPT; ++k) {
            Raw4<T> qq{hv.v[k], qxv.v[k], qyv.v[k], zv.v[k]};
            march_prims<T, SOLID>(qq, h_dry, eta[k], u[k], v[k]);
            z[k] = qq.z; hc[k] = qq.h; qxc[k] = qq.qx; qyc[k] = qq.qy;
        }
        T *stb = my_st + b * ST_B;
        stb[0] = eta[CPT - 1]; stb[NT] = u[CPT - 1]; stb[2 * NT] = v[CPT - 1]; stb[3 * NT] = z[CPT - 1];
#if TM_SPLIT_BARRIER
        mbar_arrive(&xbar[b]);                         // publishes st[b] of this row and fx[b^1] of the previous one
#endif

        // south faces of the current row = north faces of the previous one (normal velocity v)
        T g0[CPT], g1L[CPT], g1R[CPT], g2[CPT];
#pragma unroll
        for (int k = 0; k < CPT; ++k)
            face_eta<T, SOLID, true>(g, eta_p[k], v_p[k], u_p[k], z_p[k], eta[k], v[k], u[k], z[k], g0[k], g1L[k], g1R[k], g2[k]);

#if TM_SPLIT_BARRIER
        mbar_wait(&xbar[b], xpar);                     // use it/2 of xbar[b]
#else
        __syncthreads();                               // st[b] of this row and fx[b^1] of the previous one are visible
#endif
        if (warp == 0 && it + 1 + STAGES < nrows) {
            if (elect_one()) tm_issue_row<T, EDGE>(a, H, QX, QY, OCC, ring[slot], tbar, x0, y0 + it + STAGES);
        }
        sp += sizeof(RowStage<T>); op += sizeof(RowStage<T>); tbar += 1;
        if (++slot == STAGES) {
            slot = 0; tma_par ^= 1u;
            sp -= STAGES * sizeof(RowStage<T>); op -= STAGES * sizeof(RowStage<T>); tbar -= STAGES;
        }

        if (it > 0) {                                  // finish row y0 + it - 1
            const T *fe = last_thread ? &s.er[0][it - 1] : my_fx + (b ^ 1) * FX_B + 1;
            const int stride = last_thread ? MARCH_MAX_R : NT;
            const T e0 = fe[0], e1 = fe[stride], e2 = fe[2 * stride];
            // a warp whose cells of this row hold exact zeros and receive no flux writes zeros
            bool live = live_p || e0 != T(0) || e1 != T(0) || e2 != T(0) || (EDGE && (y0 + it - 1 == ny - 1 || i + CPT == nx));
#pragma unroll
            for (int k = 0; k < CPT; ++k) live = live || g0[k] != T(0) || g1L[k] != T(0) || g2[k] != T(0);
            VecN<T, CPT> ho, qxo, qyo;
#pragma unroll
            for (int k = 0; k < CPT; ++k) { ho.v[k] = qxo.v[k] = qyo.v[k] = T(0); }
            if (__any_sync(0xffffffffu, live)) {
                seg_live = true;
#pragma unroll
                for (int k = 0; k < CPT; ++k) {
                    T hn = ah[k] - dtdy * g0[k], qxn = ax[k] - dtdy * g2[k], qyn = ay[k] - dtdy * g1L[k];
                    if (k == CPT - 1) { hn -= dtdx * e0; qxn -= dtdx * e1; qyn -= dtdx * e2; }
                    if (EDGE && k == CPT - 1 && i + CPT == nx) hn += dtdx * qin * T(a.inflow[1][y0 + it - 1]);
                    if (EDGE && y0 + it - 1 == ny - 1) hn += dtdy * qin * T(a.inflow[3][i + k]);
                    if (SOLID && is_solid(z_p[k])) { hn = qxn = qyn = T(0); }
                    finish_hat2(a, dt, hn, qxn, qyn, n0_p[k], occ_p[k], lam, clamp_h, clamp_n);
                    ho.v[k] = hn; qxo.v[k] = qxn; qyo.v[k] = qyn;
                }
            }
            *reinterpret_cast<VecN<T, CPT> *>(out_h) = ho;
            *reinterpret_cast<VecN<T, CPT> *>(out_qx) = qxo;
            *reinterpret_cast<VecN<T, CPT> *>(out_qy) = qyo;
            out_h += nx; out_qx += nx; out_qy += nx;
        }
        if (it < R) {                                  // enter row y0 + it: west faces, start its accumulators
            const T *sl = first_thread ? &s.sw[0][it] : stb - 1;
            const int stride = first_thread ? MARCH_MAX_R : NT;
            T f0[CPT], f1L[CPT], f1R[CPT], f2[CPT];
            face_eta<T, SOLID, true>(g, sl[0], sl[stride], sl[2 * stride], sl[3 * stride], eta[0], u[0], v[0], z[0],
                                     f0[0], f1L[0], f1R[0], f2[0]);
#pragma unroll
            for (int k = 1; k < CPT; ++k)
                face_eta<T, SOLID, true>(g, eta[k - 1], u[k - 1], v[k - 1], z[k - 1], eta[k], u[k], v[k], z[k],
                                         f0[k], f1L[k], f1R[k], f2[k]);
            T *fxb = my_fx + b * FX_B;
            fxb[0] = f0[0]; fxb[NT] = f1L[0]; fxb[2 * NT] = f2[0];
            live_p = false;
#pragma unroll
            for (int k = 0; k < CPT; ++k) {
                ah[k] = hc[k] + dtdx * f0[k] + dtdy * g0[k];
                ax[k] = qxc[k] + dtdx * f1R[k] + dtdy * g2[k];
                ay[k] = qyc[k] + dtdx * f2[k] + dtdy * g1R[k];
                if (k < CPT - 1) { ah[k] -= dtdx * f0[k + 1]; ax[k] -= dtdx * f1L[k + 1]; ay[k] -= dtdx * f2[k + 1]; }
                if (EDGE && i + k == 0) ah[k] += dtdx * qin * T(a.inflow[0][y0 + it]);
                if (EDGE && y0 + it == 0) ah[k] += dtdy * qin * T(a.inflow[2][i + k]);
                live_p = live_p || ah[k] != T(0) || ax[k] != T(0) || ay[k] != T(0);
            }
        }
#pragma unroll
        for (int k = 0; k < CPT; ++k) {
            eta_p[k] = eta[k]; u_p[k] = u[k]; v_p[k] = v[k]; z_p[k] = z[k];
            n0_p[k] = n0_c.v[k]; occ_p[k] = a.couple ? (int)occ_c.v[k] : 0;
        }
    };

    for (int base = 0; base < nit; base += 2) {
        row(std::integral_constant<int, 0>{}, base);
        if (base + 1 < nit) row(std::integral_constant<int, 1>{}, base + 1);
        xpar ^= 1u;
    }
    }
    if (clamp_n) {
        atomicAdd(&a.ctl->clamped_volume, (double)clamp_h * (double)a.cell_area);
        atomicAdd(&a.ctl->neg_clamps, (unsigned long long)clamp_n);
    }
    // dry-segment flag of what I have just written (see flood_tmarch_kernel): exact zeros in all R rows of my
    // warp's 64 columns.  Always written, so that a stale 1 of two steps ago cannot survive.
    if (dry_out && NT / 32 == MW / 64 && (tid & 31) == 0) dry_out[warp] = seg_live ? 0 : 1;
    return lam;
}

template <typename T, int STAGES> constexpr size_t tmarch_dyn_smem() { return sizeof(RowStage<T>) * STAGES + 8 * (STAGES + 2) + 16; }

template <typename T, int CPT, int STAGES, int MINB>
__global__ void __launch_bounds__(MW / CPT, sizeof(T) == 4 ? MINB : 2) flood_tmarch_kernel(FloodArgs<T> a)
{
    pdl_enter();
    constexpr int NT = MW / CPT;
    __shared__ March2Smem<T, CPT> s;
    extern __shared__ __align__(16) unsigned char tm_dyn[];
    RowStage<T> *ring = reinterpret_cast<RowStage<T> *>(tm_dyn);
    uint64_t *bars = reinterpret_cast<uint64_t *>(tm_dyn + sizeof(RowStage<T>) * STAGES);
    const int x0 = blockIdx.x * MW, y0 = blockIdx.y * a.R;
    const int tid = threadIdx.x;
    // ---- dry chunks.  dryseg[buffer][chunk row][64-column segment] = 1: every h, qx, qy of those R x 64 cells of
    // that ping-pong buffer is an exact zero (written by this kernel only; everything else that writes flood
    // state clears the flags).  An interior chunk whose own four segments, the four above, the four below and
    // the one segment on either side are flagged at level n has zero depth on both sides of every face, so
    // every flux is zero and level n+1 is zeros too (no inflow away from the domain edge): nothing to read.
    // If its segments of the OTHER buffer (level n-1) are flagged as well, there is nothing to write either
    // and the CTA ends here.  40 % of Config 5's cells are dry; 21 % of its chunks end this way.
    // All loads of this prologue are independent (the flags of BOTH buffers are fetched, the parity picks),
    // and every warp takes the decision for itself: one memory latency, no barrier.
    const int lane = tid & 31, cy = blockIdx.y, sx0 = blockIdx.x * (MW / 64);
    int f_a = 1, f_b = 1;                              // my flag of buffer 0 / buffer 1: lanes 0..13 inputs, lanes 16..19 own segments
    if (a.dryseg) {
        size_t idx = 0; bool have = false;
        if (lane < 12) { idx = (size_t)(cy + lane / 4 - 1) * a.nsegx + sx0 + (lane & 3); have = cy > 0 && cy + 1 < (int)gridDim.y; }
        else if (lane == 12) { idx = (size_t)cy * a.nsegx + sx0 - 1; have = sx0 > 0; }
        else if (lane == 13) { idx = (size_t)cy * a.nsegx + sx0 + MW / 64; have = sx0 + MW / 64 < a.nsegx; }
        else if (lane >= 16 && lane < 16 + MW / 64) { idx = (size_t)cy * a.nsegx + sx0 + (lane - 16); have = true; }
        if (lane < 14 || (lane >= 16 && lane < 16 + MW / 64)) {
            f_a = have ? a.dryseg[idx] : 0;
            f_b = have ? a.dryseg[a.dry_stride + idx] : 0;
        }
    }
    const int path = a.chunk_flag[blockIdx.y * gridDim.x + blockIdx.x];
    const int2 hp = *reinterpret_cast<const int2 *>(&a.ctl->parity);     // parity, halt: adjacent in Ctl
    if (hp.y) return;
    uint8_t *dry_out = nullptr;
    if (a.dryseg && (path == 0 || path == 2)) {
        const int p = hp.x;
        dry_out = a.dryseg + (size_t)(p ^ 1) * a.dry_stride + (size_t)cy * a.nsegx + sx0;
        const int fin = p ? f_b : f_a, fout = p ? f_a : f_b;
        const bool in_dry = __all_sync(0xffffffffu, lane >= 14 || fin != 0);
        const bool out_dry = __all_sync(0xffffffffu, lane < 16 || lane >= 16 + MW / 64 || fout != 0);
        if (in_dry && out_dry) return;
        if (in_dry) {                                  // dried up since level n-1: write the zeros once
            const int p1 = p ^ 1;
            VecN<T, CPT> zero;
#pragma unroll
            for (int k = 0; k < CPT; ++k) zero.v[k] = T(0);
            for (int r = 0; r < a.R; ++r) {
                const size_t c = (size_t)(y0 + r) * a.nx + x0 + tid * CPT;
                *reinterpret_cast<VecN<T, CPT> *>(a.h[p1] + c) = zero;
                *reinterpret_cast<VecN<T, CPT> *>(a.qx[p1] + c) = zero;
                *reinterpret_cast<VecN<T, CPT> *>(a.qy[p1] + c) = zero;
            }
            if (tid < MW / 64) dry_out[tid] = 1;
            return;
        }
    }
    T lam = path == 1 ? march2_chunk<T, CPT, true>(a, s, x0, y0, a.R)
          : path == 3 ? tmarch_chunk<T, CPT, STAGES, true, true>(a, s, ring, bars, x0, y0, a.R, nullptr)
          : path == 2 ? tmarch_chunk<T, CPT, STAGES, true, false>(a, s, ring, bars, x0, y0, a.R, dry_out)
                      : tmarch_chunk<T, CPT, STAGES, false, false>(a, s, ring, bars, x0, y0, a.R, dry_out);
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
