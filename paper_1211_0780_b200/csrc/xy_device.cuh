// xy_device.cuh -- device-side building blocks of the XY Monte Carlo step (sm_100a).
// In-register Philox4x32-10, uniforms, fast fp32 sin/cos/atan2/exp2 with stated errors, and the
// fp64 re-evaluation of a Metropolis decision.  Shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace xyk {

// ---------------------------------------------------------------------------------------------
// Programmatic dependent launch.  The kernels of one Monte Carlo step form a chain on one stream (Metropolis pass,
// settlement, Metropolis pass, settlement, two over-relaxation passes, final reduction + exchange).  Launched with
// cudaLaunchAttributeProgrammaticStreamSerialization, a kernel's blocks may become resident while the tail of its
// predecessor still runs: they do their prologue (mbarrier set-up), then grid_dependency_wait() holds them until the
// predecessor has COMPLETED and its writes are visible -- so the data dependences are exactly those of a plain
// stream, only the launch latency and the prologue move off the critical path.  allow_dependent_launch() lets the
// successor's blocks take the multiprocessors this grid no longer fills once every block of this grid has started.
// Every kernel of the chain calls both before its first access to global memory; without the launch attribute
// both are no-ops.  XY_PDL = 0 compiles them out.
// ---------------------------------------------------------------------------------------------
#ifndef XY_PDL
#define XY_PDL 1
#endif
__device__ __forceinline__ void allow_dependent_launch() {
#if XY_PDL
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
#endif
}
__device__ __forceinline__ void grid_dependency_wait() {
#if XY_PDL
    asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
}

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11) -- north_star "generated in registers"; replaces the
// Warp Generator of P:30.  The ten round keys depend only on the seed, so the host computes
// them once and the kernels read them from the constant bank (no per-thread key schedule).
// ---------------------------------------------------------------------------------------------
struct PhiloxKeys { uint32_t k[20]; };

constexpr uint32_t kPhiloxM0 = 0xD2511F53u, kPhiloxM1 = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0 = 0x9E3779B9u, kPhiloxW1 = 0xBB67AE85u;

__host__ inline PhiloxKeys philox_round_keys(uint32_t key0, uint32_t key1) {
    PhiloxKeys K;
    for (int r = 0; r < 10; ++r) { K.k[2 * r] = key0 + r * kPhiloxW0; K.k[2 * r + 1] = key1 + r * kPhiloxW1; }
    return K;
}

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              const PhiloxKeys& K, uint32_t (&out)[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)kPhiloxM0 * c0;      // IMAD.WIDE.U32
        const uint64_t p1 = (uint64_t)kPhiloxM1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ K.k[2 * r];        // LOP3
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ K.k[2 * r + 1];
        c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// The same function with counter words 1..3 uniform over a thread block (slot, sweep number, stream):
// whatever in rounds 0-2 depends only on them is computed once per block (philox_block_invariants),
// leaving 37 instead of 40 multiplies and xors per call.  Bit-identical to philox4x32_10.
struct PhiloxInv { uint32_t j0, j1, j2, j3; };

__device__ __forceinline__ PhiloxInv philox_block_invariants(uint32_t c1, uint32_t c2, uint32_t c3, const PhiloxKeys& K) {
    PhiloxInv I;
    const uint64_t p1 = (uint64_t)kPhiloxM1 * c2;                       // round 0, uniform half
    const uint32_t i0 = (uint32_t)(p1 >> 32) ^ c1 ^ K.k[0];
    const uint32_t i1 = (uint32_t)p1;
    const uint64_t pa = (uint64_t)kPhiloxM0 * i0;                       // round 1, uniform half
    I.j0 = c3 ^ K.k[1];
    I.j1 = i1 ^ K.k[2];
    I.j2 = (uint32_t)(pa >> 32) ^ K.k[3];
    I.j3 = (uint32_t)pa ^ K.k[5];
    return I;
}

__device__ __forceinline__ void philox4x32_10_var0(uint32_t v, const PhiloxInv& I, const PhiloxKeys& K, uint32_t (&out)[4]) {
    const uint64_t q0 = (uint64_t)kPhiloxM0 * v;                        // round 0
    uint32_t c2 = (uint32_t)(q0 >> 32) ^ I.j0, c3 = (uint32_t)q0;
    const uint64_t q1 = (uint64_t)kPhiloxM1 * c2;                       // round 1
    uint32_t c0 = (uint32_t)(q1 >> 32) ^ I.j1, c1 = (uint32_t)q1;
    c2 = c3 ^ I.j2;
    {                                                                   // round 2
        const uint64_t p0 = (uint64_t)kPhiloxM0 * c0;
        const uint64_t p1 = (uint64_t)kPhiloxM1 * c2;
        c0 = (uint32_t)(p1 >> 32) ^ c1 ^ K.k[4];
        c2 = (uint32_t)(p0 >> 32) ^ I.j3;
        c1 = (uint32_t)p1; c3 = (uint32_t)p0;
    }
#pragma unroll
    for (int r = 3; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)kPhiloxM0 * c0;
        const uint64_t p1 = (uint64_t)kPhiloxM1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ K.k[2 * r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ K.k[2 * r + 1];
        c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// The same call split into its rounds, so that a kernel can interleave two calls with other work in source
// order (the rounds of one call form a serial multiply -> xor chain; see the Metropolis step of xy_sweep.cuh).
struct PhiloxState { uint32_t c0, c1, c2, c3; };

__device__ __forceinline__ void philox_var0_start(uint32_t v, const PhiloxInv& I, const PhiloxKeys& K, PhiloxState& s) {   // rounds 0..2
    const uint64_t q0 = (uint64_t)kPhiloxM0 * v;
    uint32_t c2 = (uint32_t)(q0 >> 32) ^ I.j0, c3 = (uint32_t)q0;
    const uint64_t q1 = (uint64_t)kPhiloxM1 * c2;
    uint32_t c0 = (uint32_t)(q1 >> 32) ^ I.j1, c1 = (uint32_t)q1;
    c2 = c3 ^ I.j2;
    const uint64_t p0 = (uint64_t)kPhiloxM0 * c0;
    const uint64_t p1 = (uint64_t)kPhiloxM1 * c2;
    s.c0 = (uint32_t)(p1 >> 32) ^ c1 ^ K.k[4];
    s.c2 = (uint32_t)(p0 >> 32) ^ I.j3;
    s.c1 = (uint32_t)p1; s.c3 = (uint32_t)p0;
}
template <int R>
__device__ __forceinline__ void philox_round(PhiloxState& s, const PhiloxKeys& K) {                                    // round R, 3 <= R <= 9
    const uint64_t p0 = (uint64_t)kPhiloxM0 * s.c0;
    const uint64_t p1 = (uint64_t)kPhiloxM1 * s.c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ s.c1 ^ K.k[2 * R];
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ s.c3 ^ K.k[2 * R + 1];
    s.c1 = (uint32_t)p1; s.c3 = (uint32_t)p0; s.c0 = n0; s.c2 = n2;
}

enum : uint32_t { kStreamInit = 0, kStreamMetBlack = 1, kStreamMetWhite = 2, kStreamPT = 3 };   // R12

// ---------------------------------------------------------------------------------------------
// Uniforms (R17).  u24(w) = (w >> 8) * 2^-24 is exact in fp32.  The proposal angle is
// fl32(2pi_f * u24): because 2^-24 is a power of two, (float)(w>>8) * (2pi_f * 2^-24) rounds
// once to exactly that value.
// ---------------------------------------------------------------------------------------------
constexpr float kTwoPiF = 6.2831855f;                                   // 0x40C90FDB
constexpr float kTwoPiU24 = 6.2831855f * 5.9604644775390625e-08f;       // 2pi_f * 2^-24 (exact scaling)
constexpr float kInvU24 = 5.9604644775390625e-08f;                      // 2^-24
constexpr float kPiF = 3.14159274f;
constexpr float kHalfPiF = 1.57079637f;

__device__ __forceinline__ float word_to_angle(uint32_t w) { return (float)(w >> 8) * kTwoPiU24; }
__device__ __forceinline__ float word_to_u24(uint32_t w) { return (float)(w >> 8) * kInvU24; }

// ---------------------------------------------------------------------------------------------
// Fast fp32 math.  Stated errors (measured by tests/test_gpu_parity.py::test_device_math_errors
// against fp64 on [0, 2pi]):  sin/cos abs error <= 7.5e-7 (MUFU.SIN/COS after one FMUL by 1/2pi);
// atan2 abs error <= 8e-7 rad; ex2.approx relative error <= 2^-22.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void fast_sincos(float x, float& s, float& c) {
    s = __sinf(x);
    c = __cosf(x);
}

__device__ __forceinline__ float fast_ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ float fast_rcp(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// atan2(y, x) in [0, 2pi] for (x, y) != (0, 0): octant reduction to r = min/max in [0, 1], then a
// degree-13 odd minimax polynomial (Remez fit, |error| <= 2.5e-7 in exact arithmetic).
__device__ __forceinline__ float fast_atan2_pos(float y, float x) {
    const float ax = fabsf(x), ay = fabsf(y);
    const float mx = fmaxf(ax, ay), mn = fminf(ax, ay);
    const float r = mn * fast_rcp(mx);
    const float s = r * r;
    float p = 0.006811792962253094f;
    p = fmaf(p, s, -0.0336042195558548f);
    p = fmaf(p, s, 0.07962366938591003f);
    p = fmaf(p, s, -0.1323334276676178f);
    p = fmaf(p, s, 0.19807815551757812f);
    p = fmaf(p, s, -0.3331736922264099f);
    p = fmaf(p, s, 0.9999961256980896f);
    float a = p * r;
    a = (ay > ax) ? (kHalfPiF - a) : a;
    a = (x < 0.0f) ? (kPiF - a) : a;
    a = (y < 0.0f) ? (kTwoPiF - a) : a;
    return a;
}

// ---------------------------------------------------------------------------------------------
// fp64 re-evaluation of one Metropolis decision from the STORED angles (not from the staged
// fp32 sin/cos): the definition of include/xy.h, computed in double like the paper's Eq. 1
// demands.  Taken by ~1e-4 of the decisions, so it is kept out of line.
//   other: this slot's other-colour array [z][y][W];  par: x parity of this site's row,
//   xh: x >> 1.  Neighbour order mirrors the definition: -x, -y, -z, +x, +y, +z.
// ---------------------------------------------------------------------------------------------
// fp64 sin and cos of an angle in [0, 2 pi] (the range every stored or proposed angle lies in): quadrant reduction with a
// two-part pi/2, then the Taylor polynomials to r^17 / r^16 on |r| <= pi/4 (truncation 1e-19 / 2e-18, so the result
// is within ~1.5e-16 of the true value like a libm sincos).  One third of the dependent-operation depth of the
// general-range library routine: the fp64 settlement of a close decision holds up a whole thread block (resident
// kernel) for the length of this chain.  Measured against numpy by tests/test_gpu_parity.py::test_device_math_errors.
__device__ __forceinline__ void sincos_0_2pi(double x, double& s, double& c) {
    const double kf = rint(x * 0.63661977236758134308);
    double r = fma(-kf, 1.5707963267948966, x);
    r = fma(-kf, 6.123233995736766e-17, r);
    const double z = r * r;
    double ps = 2.81145725434552060e-15, pc = 4.77947733238738525e-14;
    ps = fma(ps, z, -7.64716373181981641e-13); pc = fma(pc, z, -1.14707455977297245e-11);
    ps = fma(ps, z, 1.60590438368216133e-10);  pc = fma(pc, z, 2.08767569878681002e-09);
    ps = fma(ps, z, -2.50521083854417202e-08); pc = fma(pc, z, -2.75573192239858883e-07);
    ps = fma(ps, z, 2.75573192239858925e-06);  pc = fma(pc, z, 2.48015873015873016e-05);
    ps = fma(ps, z, -1.98412698412698413e-04); pc = fma(pc, z, -1.38888888888888894e-03);
    ps = fma(ps, z, 8.33333333333333322e-03);  pc = fma(pc, z, 4.16666666666666644e-02);
    ps = fma(ps, z, -1.66666666666666657e-01); pc = fma(pc, z, -5.00000000000000000e-01);
    const double sr = fma(r * z, ps, r), cr = fma(z, pc, 1.0);
    const int q = (int)kf;
    s = (q & 1) ? cr : sr; c = (q & 1) ? sr : cr;
    if (q & 2) s = -s;
    if ((q + 1) & 2) c = -c;
}

// The fp64 acceptance test u < exp(x), x = -beta dE, taken as log(u) < x: the logarithm does not depend on the fields,
// so it leaves the dependent chain of the settlement (callers compute it early).  Both forms agree except where u and
// exp(x) differ by a few ulp; u = 0 keeps the exp form (0 < exp(x) fails only when exp underflows to zero).
__device__ __forceinline__ double accept_log_u(double u) { return u > 0.0 ? log(u) : 0.0; }
__device__ __forceinline__ bool accept_exact(double u, double log_u, double x) { return u > 0.0 ? log_u < x : exp(x) > 0.0; }

__device__ __noinline__ bool metropolis_exact(const float* __restrict__ other, int L, int W, int par,
                                              int xh, int y, int z, float t_old, float t_new, float u,
                                              float beta32) {
    const int xm = par ? xh : (xh == 0 ? W - 1 : xh - 1);
    const int xp = par ? (xh + 1 == W ? 0 : xh + 1) : xh;
    const int ym = y == 0 ? L - 1 : y - 1, yp = y + 1 == L ? 0 : y + 1;
    const int zm = z == 0 ? L - 1 : z - 1, zp = z + 1 == L ? 0 : z + 1;
    const size_t row = (size_t)z * L + y;
    const float nb[6] = {
        other[row * W + xm], other[((size_t)z * L + ym) * W + xh], other[((size_t)zm * L + y) * W + xh],
        other[row * W + xp], other[((size_t)z * L + yp) * W + xh], other[((size_t)zp * L + y) * W + xh] };
    const double lu = accept_log_u((double)u);
    double hx = 0.0, hy = 0.0;
#pragma unroll 1
    for (int j = 0; j < 6; ++j) {
        double s, c;
        sincos_0_2pi((double)nb[j], s, c);
        hx += c; hy += s;
    }
    double so, co, sn, cn;
    sincos_0_2pi((double)t_old, so, co);
    sincos_0_2pi((double)t_new, sn, cn);
    const double dE = -(hx * (cn - co) + hy * (sn - so));
    return accept_exact((double)u, lu, -(double)beta32 * dE);
}

// Half-width of the window around p_fast inside which the decision is re-evaluated in fp64:
// window = |beta| * kWindowPerBeta + kWindowAbs.  With e_s = 7.5e-7 the stated sin/cos error, the fast
// path's g = h.(S' - S) is off by at most |dh||dS| + |h||d(dS)| <= 6 e_s * 2 sqrt2 + 2 e_s * 6 sqrt2
// = 34 e_s = 2.6e-5 plus fp32 rounding of the six-term sums and the two products (< 8e-6), so
// |p_fast - p| <= p beta |dg| < beta * 3.4e-5 for p <= 1; ex2.approx and the rounding of its argument
// add < 1e-6 relative; the fast path compares against fl32(word) * 2^-32, which is u24 up to 2^-24 = 6e-8.
// kWindowPerBeta = 4e-5 and kWindowAbs = 1.5e-6 leave a margin on all of these.
// tests/test_gpu_parity.py::test_fast_path_window measures the actual |p_fast - p_oracle|.
constexpr float kWindowPerBeta = 4.0e-5f;
constexpr float kWindowAbs = 1.5e-6f;

}  // namespace xyk
