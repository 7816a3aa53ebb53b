// flood_pk.cuh -- the fp32 arithmetic of the flood-cell update (Eq. (2); flux, sources and
// finish exactly as face_eta() / finish_hat2() of flood_march.cuh / flood_march2.cuh) on PAIRS of
// cells with Blackwell's packed single-precision instructions (FADD2 / FMUL2 / FFMA2: two IEEE
// fp32 operations per issue slot).
//
//   Why: ncu shows the flood kernel issue-bound (75 % of issue slots busy, DRAM at 45 %), with a
//   third of its instructions FADD/FMUL/FFMA.  The row-marching kernel gives every thread two
//   adjacent columns, so each of its faces and cells comes as a pair: .x = first column (or the
//   face west/south of it), .y = second.  min/max/select/compare and MUFU stay scalar per half.
//
//   Each half is computed with the same operations, in the same order, as the scalar path, with
//   the FMA contractions written out (the scalar path leaves them to the compiler).
#pragma once

#include "flood_march2.cuh"

namespace fp {

// raw conserved -> (eta, u, v) of two cells; SOLID: a solid cell (z = +inf) holds h = q = 0, eta = +inf
template <bool SOLID>
__device__ __forceinline__ void prims_x2(f2 &h, f2 &qx, f2 &qy, f2 z, float h_dry, f2 &eta, f2 &u, f2 &v)
{
    if (SOLID) {
        if (is_solid(z.x)) { h.x = qx.x = qy.x = 0.f; }
        if (is_solid(z.y)) { h.y = qx.y = qy.y = 0.f; }
    }
    const f2 r = pk(h.x > h_dry ? fast_rcp(h.x) : 0.f, h.y > h_dry ? fast_rcp(h.y) : 0.f);
    u = mul2(qx, r); v = mul2(qy, r);
    eta = add2(h, z);
}

// two faces at once; VOTE as in face_eta(): a warp none of whose faces is wet skips the flux.
// SOLID: a solid side is replaced by the wall ghost of the other side (C13, C16), as in face_eta().
template <bool SOLID>
__device__ __forceinline__ void face_eta_x2(float g, f2 etaL, f2 uL, f2 vL, f2 zL, f2 etaR, f2 uR, f2 vR, f2 zR,
                                            f2 &f0, f2 &f1L, f2 &f1R, f2 &f2_)
{
    if (SOLID) {
        const bool l0 = is_solid(zL.x), l1 = is_solid(zL.y);
        if (l0) { etaL.x = etaR.x; uL.x = -uR.x; vL.x = vR.x; zL.x = zR.x; }
        if (l1) { etaL.y = etaR.y; uL.y = -uR.y; vL.y = vR.y; zL.y = zR.y; }
        const bool r0 = is_solid(zR.x), r1 = is_solid(zR.y);
        if (r0) { etaR.x = etaL.x; uR.x = -uL.x; vR.x = vL.x; zR.x = zL.x; }
        if (r1) { etaR.y = etaL.y; uR.y = -uL.y; vR.y = vL.y; zR.y = zL.y; }
    }
    const f2 zf = max2(zL, zR);
    const f2 hL = max2(pk1(0.f), sub2(etaL, zf));
    const f2 hR = max2(pk1(0.f), sub2(etaR, zf));
    const bool wet = fmaxf(fmaxf(hL.x, hR.x), fmaxf(hL.y, hR.y)) > 0.f;
    if (!__any_sync(0xffffffffu, wet)) { f0 = f1L = f1R = f2_ = pk1(0.f); return; }
    const f2 ghL = mul2(hL, pk1(g)), ghR = mul2(hR, pk1(g));
    const f2 cL = sqrt2(ghL), cR = sqrt2(ghR);
    const f2 tL = fma2(cR, pk1(-2.f), uR), tR = fma2(cL, pk1(2.f), uL);
    const f2 uLe = pk(hL.x > 0.f ? uL.x : tL.x, hL.y > 0.f ? uL.y : tL.y);
    const f2 uRe = pk(hR.x > 0.f ? uR.x : tR.x, hR.y > 0.f ? uR.y : tR.y);
    const f2 us = fma2(add2(uLe, uRe), pk1(0.5f), sub2(cL, cR));
    const f2 cs = fma2(add2(cL, cR), pk1(0.5f), mul2(sub2(uLe, uRe), pk1(0.25f)));
    const f2 a1 = sub2(uLe, cL), a2 = sub2(us, cs), b1 = add2(uRe, cR), b2 = add2(us, cs);
    const f2 sL = pk(fminf(fminf(a1.x, a2.x), 0.f), fminf(fminf(a1.y, a2.y), 0.f));
    const f2 sR = pk(fmaxf(fmaxf(b1.x, b2.x), 0.f), fmaxf(fmaxf(b1.y, b2.y), 0.f));
    const f2 qL = mul2(hL, uLe), qR = mul2(hR, uRe);
    const f2 mL = mul2(qL, uLe), mR = mul2(qR, uRe);
    // both products rounded before the difference: equal depths give de = 0 exactly (lake at rest)
    const f2 de = mul2(sub2(mul2(ghR, hR), mul2(ghL, hL)), pk1(0.5f));
    const f2 den = max2(sub2(sR, sL), pk1(1e-30f));
    const f2 w = mul2(neg2(sL), rcp2(den));
    const f2 dq = sub2(qR, qL);
    f0 = fma2(w, fma2(neg2(sR), sub2(hR, hL), dq), qL);
    f1L = fma2(w, fma2(neg2(sR), dq, add2(sub2(mR, mL), de)), mL);
    f1R = sub2(f1L, de);
    f2_ = mul2(f0, pk(f0.x >= 0.f ? vL.x : vR.x, f0.y >= 0.f ? vL.y : vR.y));
}

// clamp (C12), Manning friction (C6), wave speed of the new state for two cells
__device__ __forceinline__ void finish_hat_x2(const FloodArgs<float> &a, float dt, f2 &hn, f2 &qxn, f2 &qyn, f2 n0,
                                              int np0, int np1, float &lam, float &clamp_h, int &clamp_n)
{
    clamp_h += (hn.x < 0.f ? -hn.x : 0.f) + (hn.y < 0.f ? -hn.y : 0.f);
    clamp_n += (hn.x < 0.f ? 1 : 0) + (hn.y < 0.f ? 1 : 0);
    hn = max2(hn, pk1(0.f));
    const bool wet0 = hn.x > a.h_dry, wet1 = hn.y > a.h_dry;
    const f2 hs = max2(hn, pk1(a.h_dry));
    const f2 n = a.couple ? mul2(n0, pk(1.f + float(min(np0, a.n_cap)), 1.f + float(min(np1, a.n_cap)))) : n0;
    const f2 sq = sqrt2(fma2(qxn, qxn, mul2(qyn, qyn)));
    const f2 pw = pk(pow_m73(hs.x), pow_m73(hs.y));
    const f2 D = fma2(mul2(mul2(mul2(mul2(pk1(dt), pk1(a.g)), n), n), sq), pw, pk1(1.f));
    const f2 rD = pk(wet0 ? fast_rcp(D.x) : 0.f, wet1 ? fast_rcp(D.y) : 0.f);
    qxn = mul2(qxn, rD); qyn = mul2(qyn, rD);
    const f2 rh = rcp2(hs), c = sqrt2(mul2(hs, pk1(a.g)));
    const f2 ux = mul2(qxn, rh), uy = mul2(qyn, rh);
    const f2 lx = mul2(add2(pk(fabsf(ux.x), fabsf(ux.y)), c), pk1(a.inv_dx));
    const f2 ly = mul2(add2(pk(fabsf(uy.x), fabsf(uy.y)), c), pk1(a.inv_dy));
    const float l0 = wet0 ? fmaxf(lx.x, ly.x) : 0.f, l1 = wet1 ? fmaxf(lx.y, ly.y) : 0.f;
    lam = fmaxf(lam, fmaxf(l0, l1));
}

}  // namespace fp
