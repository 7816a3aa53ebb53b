// common.cuh -- device-side control block and small helpers shared by the kernels of
// libfloodped.so.  (Nothing here is shared with oracle/: the oracle is a separate C program.)
#pragma once

#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

namespace fp {

// Everything that changes from step to step and must not round-trip through the host
// (the CFL time step is global and adaptive; north_star: "no host round-trip").
// One instance lives in device memory; kernels of a step read it, the tail kernel advances it.
struct Ctl {
    double t, dt;                    // time reached; dt of the step being taken
    double t_end, dt_max, cfl;
    double q_in;                     // inflow per unit width for the step being taken, m2/s
    double clamped_volume;           // C12 accounting
    unsigned long long lam_bits;     // bits of max over wet cells of (|u|+c)/dx, (|v|+c)/dy at n+1
    unsigned long long neg_clamps;
    long long step, deposits;
    int parity;                      // which of the two flood buffers holds level n
    int halt;                        // t >= t_end: every kernel of the step returns at once
    int D;                           // sandbag deposits of the step being taken
    int cursor, layer, bags, complete;
    unsigned int scan_epoch;         // makes the look-back flags of the scan self-resetting
    unsigned int scan_ticket;        // dynamic tile index of the scan
    int occ_next;                    // N_p buffer the binning chain of the NEXT step fills (= parity ^ 1), published by the pedestrian step
    // SURVEY 8f-3 (D1-D9)
    double outflow_volume;           // volume that left through open edges (D1)
    long long spawned;               // newcomers let in by the doors so far (D3); also the Philox counter (D5)
    int triggered;                   // a wet cell has been seen: no more entries, everybody evacuates (D7)
    float pair_c1, pair_c2;          // fp32 pair force A_s e^{(2r-d)/B_s} = 2^{c1 + c2 d}: read from memory once per thread so that they
                                     // stay in registers (as kernel parameters ptxas reloads them from the constant bank per candidate)
};

template <typename T> struct Vec4 { T v[4]; };
template <> struct __align__(16) Vec4<float> { float v[4]; };
template <> struct __align__(32) Vec4<double> { double v[4]; };

// N adjacent reals moved with one 64- or 128-bit access
template <typename T, int N> struct __align__(sizeof(T) * N) VecN { T v[N]; };

template <typename T> __device__ __forceinline__ T solid_z();
template <> __device__ __forceinline__ float solid_z<float>() { return CUDART_INF_F; }
template <> __device__ __forceinline__ double solid_z<double>() { return CUDART_INF; }

__device__ __forceinline__ bool is_solid(float z) { return z == CUDART_INF_F; }
__device__ __forceinline__ bool is_solid(double z) { return z == CUDART_INF; }

// correctly rounded single operations (never contracted into FMA): the integer-valued
// decisions of the pedestrian step are taken with these so that they are reproducible
// bit for bit by a float replay on the CPU
__device__ __forceinline__ float  mul_rn(float a, float b)   { return __fmul_rn(a, b); }
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ float  add_rn(float a, float b)   { return __fadd_rn(a, b); }
__device__ __forceinline__ double add_rn(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ float  div_rn(float a, float b)   { return __fdiv_rn(a, b); }
__device__ __forceinline__ double div_rn(double a, double b) { return __ddiv_rn(a, b); }

// Approximate single-instruction math (MUFU) for the flood kernel's fp32 path: relative error
// <= 2^-22, far inside the 1e-5 tolerance of the fp32 configs; fp64 stays IEEE.
__device__ __forceinline__ float  fast_rcp(float a)  { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }
__device__ __forceinline__ double fast_rcp(double a) { return 1.0 / a; }
__device__ __forceinline__ float  fast_sqrt(float a)  { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }
__device__ __forceinline__ double fast_sqrt(double a) { return sqrt(a); }
__device__ __forceinline__ float  fast_rsqrt(float a)  { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }
__device__ __forceinline__ double fast_rsqrt(double a) { return rsqrt(a); }
__device__ __forceinline__ float  fast_exp(float a)
{
    float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a * 1.4426950408889634f)); return r;
}
__device__ __forceinline__ double fast_exp(double a) { return exp(a); }
// h^(-7/3) for the Manning term, h > h_dry > 0
__device__ __forceinline__ float  pow_m73(float h)
{
    float l, r;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(l) : "f"(h));
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(l * -2.3333333333333335f));
    return r;
}
__device__ __forceinline__ double pow_m73(double h) { return 1.0 / (h * h * cbrt(h)); }
__device__ __forceinline__ float  real_sqrt(float a)  { return sqrtf(a); }
__device__ __forceinline__ double real_sqrt(double a) { return sqrt(a); }

// ---- Blackwell packed single precision (FADD2 / FMUL2 / FFMA2: two IEEE fp32 operations per issue
// slot) on pairs; min/max/select/compare and MUFU stay scalar per half
typedef float2 f2;

__device__ __forceinline__ f2 pk(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ f2 pk1(float a) { return make_float2(a, a); }
__device__ __forceinline__ f2 neg2(f2 a) { return make_float2(-a.x, -a.y); }          // folds into an operand modifier
__device__ __forceinline__ f2 add2(f2 a, f2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ f2 sub2(f2 a, f2 b) { return __fadd2_rn(a, neg2(b)); }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ f2 max2(f2 a, f2 b) { return make_float2(fmaxf(a.x, b.x), fmaxf(a.y, b.y)); }
__device__ __forceinline__ f2 sqrt2(f2 a) { return make_float2(fast_sqrt(a.x), fast_sqrt(a.y)); }
__device__ __forceinline__ f2 rcp2(f2 a) { return make_float2(fast_rcp(a.x), fast_rcp(a.y)); }

// Programmatic dependent launch: a kernel launched with the programmatic-serialization attribute
// may start while the kernel before it in the stream is still draining; everything it reads from
// that kernel must come after this wait (a no-op for ordinary launches).
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
// Let the next kernel of the stream be scheduled now: its CTAs then sit at their pdl_wait() until
// this grid has completed and flushed, instead of being launched after it (saves the launch gap).
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_enter() { pdl_trigger(); pdl_wait(); }

__device__ __forceinline__ void atomic_max_lambda(Ctl *ctl, double lam)
{
    // lam >= 0: the IEEE bit pattern of non-negative doubles is ordered like the integers
    atomicMax(&ctl->lam_bits, (unsigned long long)__double_as_longlong(lam));
}

}  // namespace fp
