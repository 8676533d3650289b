// dt_orbit.cuh -- fp64 device arithmetic of kernel 1: per-orbit precompute, Kepler solves (cold and
// warm-started), heliocentric position, conservative pre-cull, gnomonic projection.
//
// Definitions follow DESIGN.md "What the path computes" (BASELINE.json north_star; the paper's
// skeleton is PAPER.md:202 "converting the set of orbital parameters into a sky position at the
// time of each image and converting these celestial coordinates to locations within the pixel
// grid").  Formulation notes (all differ from the CPU oracle on purpose -- no shared code):
//   * the orbit basis is pre-rotated to the equatorial frame and pre-scaled: r_eq = A (cosE - e)
//     + B sinE with A = a R_eps P, B = a sqrt(1-e^2) R_eps Q, so steps "subtract observer" and
//     "rotate ecliptic -> equatorial" commute into the per-orbit / per-exposure constants;
//   * the projection is the VECTOR form xi = q.e_E / q.t, eta = q.e_N / q.t;
//   * the Kepler state is carried as u = E - M with (sin E, cos E) and advanced from exposure to
//     exposure by a 4th-order series step + rotation by Taylor (sin, cos) + one Newton polish,
//     falling back to a libdevice-sincos Newton solve from a monotone start when the step is large.
#pragma once

#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

namespace dt {

constexpr double kPi = 3.14159265358979323846;
constexpr double kTwoPiHi = 6.28318530717958623200;     // fl(2 pi)
constexpr double kTwoPiLo = 2.44929359829470641435e-16;  // 2 pi - fl(2 pi)
constexpr double kInvTwoPi = 0.15915494309189534561;

struct Orbit {
    double n, e, M0;
    double Ax, Ay, Az, Bx, By, Bz;  // equatorial, AU
    double cos2_cull;               // cos^2 of the pre-cull cone half-angle
    double rho2_close;              // pairs closer than this (AU^2) are always refined
    double vmax;                    // perihelion speed, AU / day (the largest speed on the orbit)
    double inv_n;                   // 1 / n
    bool valid;
};

__device__ __forceinline__ bool orbit_valid(const double el[6])
{
    bool fin = isfinite(el[0]) && isfinite(el[1]) && isfinite(el[2]) && isfinite(el[3]) &&
               isfinite(el[4]) && isfinite(el[5]);
    return fin && el[0] > 0.0 && el[1] >= 0.0 && el[1] < 1.0;
}

// Per-orbit precompute (hot-path step 1).  tan_fov: tan of the footprint half-diagonal.
__device__ __forceinline__ Orbit orbit_setup(const double el_in[6], double gm, double cos_eps,
                                             double sin_eps, double inv_c, double tan_fov)
{
    Orbit o;
    double el[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) el[k] = el_in[k];
    o.valid = orbit_valid(el);
    if (!o.valid) { el[0] = 1.0; el[1] = 0.0; el[2] = el[3] = el[4] = el[5] = 0.0; }
    const double a = el[0], e = el[1];
    o.n = sqrt(gm / (a * a * a));
    o.inv_n = 1.0 / o.n;
    o.e = e;
    o.M0 = el[5];
    double si, ci, sO, cO, sw, cw;
    sincos(el[2], &si, &ci);
    sincos(el[3], &sO, &cO);
    sincos(el[4], &sw, &cw);
    // perifocal basis in the ecliptic frame
    const double Px = cO * cw - sO * sw * ci, Py = sO * cw + cO * sw * ci, Pz = sw * si;
    const double Qx = -cO * sw - sO * cw * ci, Qy = -sO * sw + cO * cw * ci, Qz = cw * si;
    const double b = a * sqrt(1.0 - e * e);
    // rotate to equatorial: y' = y cos(eps) - z sin(eps), z' = y sin(eps) + z cos(eps)
    o.Ax = a * Px;
    o.Ay = a * (Py * cos_eps - Pz * sin_eps);
    o.Az = a * (Py * sin_eps + Pz * cos_eps);
    o.Bx = b * Qx;
    o.By = b * (Qy * cos_eps - Qz * sin_eps);
    o.Bz = b * (Qy * sin_eps + Qz * cos_eps);
    // pre-cull cone: footprint half-diagonal + the largest angle light-time can move the object as
    // seen by the observer, asin(v_max / c) with v_max the perihelion speed (|r(t) - r(t - tau)| <=
    // v_max tau and tau = rho0 / c exactly, so the bound does not depend on rho0), + slack.
    const double vmax = sqrt(gm / a * (1.0 + e) / (1.0 - e));
    o.vmax = vmax;
    // The 1e-4 rad of slack for the cull-quality Kepler chain (below) was derived and validated for e <= 0.9 (its
    // truncation grows like e / (1 - e)); no cone for more eccentric orbits: they are refined everywhere.
    const double th = (e > 0.9) ? 2.0 : atan(tan_fov) * 1.01 + 1.05 * asin(fmin(vmax * inv_c, 1.0)) + 1.4e-4;
    const double cth = (th < 1.5) ? cos(th) : 0.0;
    o.cos2_cull = (th < 1.5) ? cth * cth : 0.0;
    // The cull may run on an UNPOLISHED order-2 Kepler state, off by <= 6e-6 rad in E (k_propagate), i.e.
    // by <= 6e-6 a AU in position (|dr/dE| <= a) and 6e-6 a / rho in direction: 1e-4 rad of the slack
    // above are reserved for it, which holds for rho >= 0.06 a; closer pairs (and anything inside
    // 0.1 AU) are refined unconditionally.
    // (a cone wider than 1.5 rad is no cone: such an orbit is refined everywhere -- through an infinite rho2_close,
    // which costs the hot loop no compare of its own)
    o.rho2_close = (th < 1.5) ? fmax(0.01, 0.0036 * a * a) : INFINITY;
    return o;
}

// ---- small fp64 helpers: MUFU seed + Newton, no slow-path branches ---------------------------------
// 1/x for normal, finite x; measured on B200: MUFU seed 9.8e-7 relative, 9.7e-13 after one
// iteration, correctly rounded after two.
template <int ITERS>
__device__ __forceinline__ double rcp_nr(double x)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
#pragma unroll
    for (int i = 0; i < ITERS; ++i) {
        double e = fma(-x, r, 1.0);
        r = fma(r, e, r);
    }
    return r;
}

// sqrt(a) for normal a > 0; Goldschmidt iterations from the MUFU rsqrt seed.
template <int ITERS>
__device__ __forceinline__ double sqrt_nr(double a)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    double g = a * y, h = 0.5 * y;
#pragma unroll
    for (int i = 0; i < ITERS; ++i) {
        double r = fma(-g, h, 0.5);
        g = fma(g, r, g);
        h = fma(h, r, h);
    }
    return g;
}

// Polynomial coefficients of the hot warm step live in constant memory: an FP64 instruction can take
// a constant-bank operand directly, whereas a 64-bit literal that is not a short immediate costs two
// move instructions per use (r1b profile: 33 UMOV / IMAD.MOV per pair, a quarter of all issued
// instructions).
__constant__ double kWarmC[16] = {
    1.0 / 6.0,        // 0: a3 scale, -sin coefficient
    1.0 / 12.0,       // 1
    5.0,              // 2
    1.0 / 120.0,      // 3
    1.0 / 5040.0,     // 4
    1.0 / 362880.0,   // 5
    1.0 / 24.0,       // 6
    1.0 / 720.0,      // 7
    1.0 / 40320.0,    // 8
    0.04,             // 9: |x| bound
    0.01,             // 10: |x a2| bound
    0.015,            // 11, 12: ORDER 3 bounds
    0.004,
    0.003,            // 13, 14: ORDER 2 bounds
    0.001,
    0.0};

// ---- Kepler state ----------------------------------------------------------------------------------
// E = M + u (unreduced), s = sin E, c = cos E.  |u| <= e < 1, so u keeps full absolute precision
// however large M is, and the residual E - e sin E - M = u - e s has no cancellation against M.
struct Kepler {
    double M, u, s, c;
};

// Cold solve: reduce M to m in [-pi, pi], fold to [0, pi], start at E0 = min(m + e, pi) (f convex on
// [0, pi] with f(E0) >= 0, so Newton descends monotonically), Newton with libdevice sincos until
// every lane of the warp has |dE| < 2e-9 (then the last first-order update is exact to ~1e-17).
// Must be called by all 32 lanes of the warp.
__device__ __forceinline__ Kepler kepler_cold(double e, double M)
{
    const double k = rint(M * kInvTwoPi);
    double m = fma(-k, kTwoPiHi, M);
    m = fma(-k, kTwoPiLo, m);
    const double sg = (m < 0.0) ? -1.0 : 1.0;
    m = fabs(m);
    double E = fmin(m + e, kPi);
    double s, c, dE;
    bool done = false;
    for (int it = 0; it < 60; ++it) {
        sincos(E, &s, &c);
        const double f = fma(-e, s, E) - m;
        const double g = fma(-e, c, 1.0);
        dE = f / g;
        if (!done) E -= dE; else dE = 0.0;
        done = done || (fabs(dE) < 2e-9);
        if (__all_sync(0xffffffffu, done)) break;
    }
    // sin/cos were taken at E + dE: first-order update to the final E (dE^2/2 < 2e-18)
    const double s1 = fma(-dE, c, s), c1 = fma(dE, s, c);
    Kepler K;
    K.M = M;
    K.u = sg * (E - m);
    K.s = sg * s1;
    K.c = c1;
    return K;
}

// Newton from a nearby state toward a new mean anomaly with libdevice sincos ("reference" mode of
// the light-time re-solve).  Works on u directly: f = u - e sin(M + u).  All 32 lanes must call.
__device__ __forceinline__ Kepler kepler_newton_from(double e, const Kepler &K0, double Mn)
{
    const double dM = Mn - K0.M;
    // E_old = M_old + u_old; new equation: (E_old + th) - e sin(E_old + th) = M_old + dM
    double th = 0.0, s = K0.s, c = K0.c, d;
    const double f00 = fma(-e, K0.s, K0.u) - dM;  // residual at th = 0
    bool done = false;
    // sin(E_old + th) by rotating (s0, c0) with libdevice sincos(th): th is small but arbitrary
    for (int it = 0; it < 60; ++it) {
        double st, ct;
        sincos(th, &st, &ct);
        s = fma(K0.s, ct, K0.c * st);
        c = fma(K0.c, ct, -K0.s * st);
        const double f = fma(-e, s - K0.s, f00 + th);
        const double g = fma(-e, c, 1.0);
        d = f / g;
        if (!done) th -= d; else d = 0.0;
        done = done || (fabs(d) < 2e-9);
        if (__all_sync(0xffffffffu, done)) break;
    }
    Kepler K;
    K.M = Mn;
    K.u = K0.u + (th - dM);
    K.s = fma(-d, c, s);
    K.c = fma(d, s, c);
    return K;
}

// Warm step: series reversion of f(th) = f0 + g th + (e s/2) th^2 + (e c/6) th^3 - (e s/24) th^4 = 0
// to 4th order, rotation of (s, c) by th with Taylor sin/cos (|th| <= 0.05: next terms < 3e-20),
// then one Newton polish with a refined reciprocal.  `ok` is false when the step is outside the
// domain where the truncated series is accurate enough for the polish to reach full precision;
// the caller then falls back to kepler_cold.
// The step comes in three orders of the series / Taylor polynomials, chosen warp-uniformly from the
// first-order step x (accuracy of (u, sin E, cos E) against 40-digit solutions, e <= 0.9):
//   ORDER 4: |x| <= 0.04,  |x a2| <= 0.01    (worst 1.8e-13)   the general exposure-to-exposure step
//   ORDER 3: |x| <= 0.015, |x a2| <= 0.004   (worst 2.4e-15)   what main-belt cadences need: 7 fewer
//                                                               FP64 instructions
//   ORDER 2: |x| <= 0.003, |x a2| <= 0.001   (worst 5.9e-16)   the light-time re-solve (x ~ n tau):
//                                                               13 fewer
// One Newton step on the carried state: f = u - e s, 1/g from its own MUFU seed + one Newton step
// (1e-12 relative, measured).  One Newton step from the previous 1/g instead leaves ((g1 - g)/g)^2 of
// the correction behind, up to 1.3e-10 rad at e = 0.9 next to a perihelion.
__device__ __forceinline__ Kepler kepler_polish(double e, const Kepler &K0)
{
    const double f1 = fma(-e, K0.s, K0.u);
    const double g1 = fma(-e, K0.c, 1.0);
    const double d = -f1 * rcp_nr<1>(g1);
    Kepler K;
    K.M = K0.M;
    K.u = K0.u + d;
    K.s = fma(d, K0.c, K0.s);
    K.c = fma(-d, K0.s, K0.c);
    return K;
}

// Two Newton steps on a state that may be off by up to ~1e-5 rad (an unpolished ORDER 2 step): the
// first with a correctly rounded reciprocal and a third-order rotation by its correction d (d^4/24 <
// 1e-21), the second first-order (d2 ~ a2 d^2 <= 1e-10).
__device__ __forceinline__ Kepler kepler_polish2(double e, const Kepler &K0)
{
    const double g1 = fma(-e, K0.c, 1.0);
    const double d = -fma(-e, K0.s, K0.u) * rcp_nr<2>(g1);
    const double d2h = 0.5 * d * d;                              // 1 - cos d
    const double sd = fma(-d * d2h, 1.0 / 3.0, d);               // sin d = d - d^3/6
    Kepler K;
    K.M = K0.M;
    K.u = K0.u + d;
    K.s = K0.s + fma(K0.c, sd, -K0.s * d2h);
    K.c = K0.c - fma(K0.s, sd, K0.c * d2h);
    return kepler_polish(e, K);
}

// POLISH = false returns the state right after the series step and the rotation: a self-consistent
// point (s = sin(M + u), c = cos(M + u)) whose u is off by the series truncation (<= 6.5e-8 rad for
// ORDER 3, <= 4.3e-6 rad for ORDER 2 inside the ORDER 3 domain, chained steps included: the next step's series starts from the exact residual of the
// state it is given, so the error does not accumulate).  Good enough to CULL with; kepler_polish
// finishes the job for the pairs that survive.
template <int ORDER, bool POLISH = true>
__device__ __forceinline__ Kepler kepler_warm_tail(double e, const Kepler &K0, double Mn, double dM, double es,
                                                   double ec, double rg, double x, double a2)
{
    const double *C = kWarmC;
    double th;
    if (ORDER >= 3) {
        const double a3 = C[0] * ec * rg;
        // a4 = -a2 / 12;  th = x - a2 x^2 + (2 a2^2 - a3) x^3 + (5 a2 a3 - a4 - 5 a2^3) x^4
        const double a22 = a2 * a2;
        const double k3 = fma(2.0, a22, -a3);
        if (ORDER >= 4) {
            const double k4 = fma(a2, fma(C[2], a3, C[1]), -C[2] * a22 * a2);
            th = x * fma(x, fma(x, fma(x, k4, k3), -a2), 1.0);
        } else {
            th = x * fma(x, fma(x, k3, -a2), 1.0);
        }
    } else {
        th = x * fma(-x, a2, 1.0);
    }
    // Taylor rotation (sin th, cos th - 1)
    const double z = th * th;
    double ps, pc;
    if (ORDER >= 4) {
        ps = fma(z, fma(z, fma(z, C[5], -C[4]), C[3]), -C[0]);
        pc = fma(z, fma(z, fma(z, C[8], -C[7]), C[6]), -0.5);
    } else if (ORDER == 3) {
        ps = fma(z, fma(z, -C[4], C[3]), -C[0]);
        pc = fma(z, fma(z, -C[7], C[6]), -0.5);
    } else {
        ps = fma(z, C[3], -C[0]);
        pc = fma(z, C[6], -0.5);
    }
    const double st = fma(th * z, ps, th);
    const double cm = z * pc;
    const double s1 = fma(K0.s, cm, fma(K0.c, st, K0.s));
    const double c1 = fma(K0.c, cm, fma(-K0.s, st, K0.c));
    const double u1 = K0.u + (th - dM);
    Kepler K;
    K.M = Mn;
    K.u = u1;
    K.s = s1;
    K.c = c1;
    return POLISH ? kepler_polish(e, K) : K;
}

// The part of the warm step that comes before its order is known: first-order step x and a2.
struct WarmPre {
    double dM, es, ec, rg, x, a2, ax, axa2;
};
// `seed_only` (warp-uniform): 1/g straight from the MUFU seed (1e-6 relative, i.e. <= 3e-7 rad of
// theta): enough for a cull-quality step.
__device__ __forceinline__ WarmPre kepler_warm_pre(double e, const Kepler &K0, double Mn, bool seed_only = false)
{
    WarmPre w;
    w.dM = Mn - K0.M;
    w.es = e * K0.s;
    w.ec = e * K0.c;
    const double f0 = (K0.u - w.es) - w.dM;
    // full steps: one Newton iteration, 1e-12 relative (the polish removes what that costs theta)
    w.rg = seed_only ? rcp_nr<0>(1.0 - w.ec) : rcp_nr<1>(1.0 - w.ec);
    w.x = -f0 * w.rg;
    w.a2 = 0.5 * w.es * w.rg;
    w.ax = fabs(w.x);
    w.axa2 = fabs(w.x * w.a2);
    return w;
}
template <int ORDER>
__device__ __forceinline__ bool kepler_warm_in_domain(const WarmPre &w)
{
    const double *C = kWarmC;
    if (ORDER == 4) return (w.ax <= C[9]) && (w.axa2 <= C[10]);
    if (ORDER == 3) return (w.ax <= C[11]) && (w.axa2 <= C[12]);
    return (w.ax <= C[13]) && (w.axa2 <= C[14]);
}
template <int ORDER, bool POLISH = true>
__device__ __forceinline__ Kepler kepler_warm_finish(double e, const Kepler &K0, double Mn, const WarmPre &w)
{
    return kepler_warm_tail<ORDER, POLISH>(e, K0, Mn, w.dM, w.es, w.ec, w.rg, w.x, w.a2);
}

// LOW = 3 for the exposure-to-exposure step, 2 for the light-time re-solve: the warp takes the cheaper
// order when every lane's step is inside its domain (one vote), else ORDER 4.  All 32 lanes must call.
// One Newton step on a seed-quality reciprocal (1e-6 -> 1e-12) and the quantities derived from it: an ORDER 4
// series (steps up to 0.04 rad) steered by the bare seed would leave 7e-15 rad after the polish at e = 0.9.
__device__ __forceinline__ void warm_refine_rg(WarmPre &w)
{
    const double g = 1.0 - w.ec;
    const double f0 = -w.x * g;                          // x = -f0 rg with the seed rg ~ 1/g
    w.rg = w.rg * fma(-g, w.rg, 2.0);
    w.x = -f0 * w.rg;
    w.a2 = 0.5 * w.es * w.rg;
}

// The series of a POLISHED step is steered by the MUFU seed of 1/g alone (1e-6 relative: theta is off by
// <= 1e-6 |x| <= 1.5e-8 rad in the ORDER <= 3 domains, of which the Newton polish -- with its own refined
// reciprocal -- leaves a2 (1.5e-8)^2 < 1e-15); the ORDER 4 domain refines the reciprocal first.
template <int LOW>
__device__ __forceinline__ Kepler kepler_warm(double e, const Kepler &K0, double Mn, bool &ok)
{
    WarmPre w = kepler_warm_pre(e, K0, Mn, true);
    if (__all_sync(0xffffffffu, kepler_warm_in_domain<LOW>(w))) {
        ok = true;
        return kepler_warm_finish<LOW>(e, K0, Mn, w);
    }
    warm_refine_rg(w);
    ok = kepler_warm_in_domain<4>(w);
    return kepler_warm_finish<4>(e, K0, Mn, w);
}

// Wide warm step: the same 4th-order series start, but for steps 7.5 times longer (|x| <= 0.3,
// |x a2| <= 0.08, |a3| x^2 <= 0.02 -- the cubic coefficient matters at a perihelion, where a2 = 0).
// The series then leaves an error eps up to ~1e-3 in theta, so
//   * the (sin, cos) rotation polynomials carry two more terms each (|theta| <= 0.35: neglected
//     theta^15/15!, theta^14/14! < 5e-18),
//   * the first Newton polish uses a freshly refined 1/g1 (g changes by tens of per cent over such a
//     step) and rotates (s, c) by its correction d to third order (d^4/24 < 1e-20),
//   * a second, first-order polish (d2 <= ~3e-7, d2^2/2 < 1e-13 x a2) finishes the job.
// Worst error of (u, sin E, cos E) against 40-digit solutions over 2e4 accepted random steps with
// e <= 0.9: 6.5e-16 (the narrow step, with its single polish: 1.8e-13).
// ~75 FP64 instructions against ~45 for the narrow step and several hundred for a cold solve.
// POLISH2 = false stops after the first polish: <= 5.3e-8 rad in E over chained steps (cull quality).
template <bool POLISH2 = true>
__device__ __forceinline__ Kepler kepler_warm_wide_finish(double e, const Kepler &K0, double Mn, const WarmPre &w,
                                                          bool &ok)
{
    const double dM = w.dM, rg = w.rg, x = w.x, a2 = w.a2;
    const double a3 = (1.0 / 6.0) * w.ec * rg;
    const double a22 = a2 * a2;
    const double k3 = fma(2.0, a22, -a3);
    const double k4 = fma(a2, fma(5.0, a3, 1.0 / 12.0), -5.0 * a22 * a2);
    const double th = x * fma(x, fma(x, fma(x, k4, k3), -a2), 1.0);
    ok = (w.ax <= 0.3) && (w.axa2 <= 0.08) && (fabs(a3) * x * x <= 0.02);
    // Taylor rotation by th, sin to th^13, cos to th^12
    const double z = th * th;
    const double ps = fma(z, fma(z, fma(z, fma(z, fma(z, 1.0 / 6227020800.0, -1.0 / 39916800.0), 1.0 / 362880.0),
                                        -1.0 / 5040.0), 1.0 / 120.0), -1.0 / 6.0);
    const double pc = fma(z, fma(z, fma(z, fma(z, fma(z, 1.0 / 479001600.0, -1.0 / 3628800.0), 1.0 / 40320.0),
                                        -1.0 / 720.0), 1.0 / 24.0), -0.5);
    const double st = fma(th * z, ps, th);   // sin th
    const double cm = z * pc;                // cos th - 1
    const double s1 = K0.s + fma(K0.c, st, K0.s * cm);
    const double c1 = K0.c + fma(-K0.s, st, K0.c * cm);
    const double u1 = K0.u + (th - dM);
    // polish 1: fresh reciprocal, third-order rotation by d
    const double g1 = fma(-e, c1, 1.0);
    const double rg1 = rcp_nr<2>(g1);
    const double d = -fma(-e, s1, u1) * rg1;
    const double d2h = 0.5 * d * d;                              // 1 - cos d
    const double sd = fma(-d * d2h, 1.0 / 3.0, d);               // sin d = d - d^3/6
    const double s2 = s1 + fma(c1, sd, -s1 * d2h);
    const double c2 = c1 - fma(s1, sd, c1 * d2h);
    const double u2 = u1 + d;
    if (!POLISH2) {
        Kepler Kc;
        Kc.M = Mn;
        Kc.u = u2;
        Kc.s = s2;
        Kc.c = c2;
        return Kc;
    }
    // polish 2: first order, 1/g2 by one Newton step from 1/g1
    const double g2 = fma(-e, c2, 1.0);
    const double rg2 = rg1 * fma(-g2, rg1, 2.0);
    const double dd = -fma(-e, s2, u2) * rg2;
    Kepler K;
    K.M = Mn;
    K.u = u2 + dd;
    K.s = fma(dd, c2, s2);
    K.c = fma(-dd, s2, c2);
    return K;
}

template <bool POLISH2 = true>
__device__ __forceinline__ Kepler kepler_warm_wide(double e, const Kepler &K0, double Mn, bool &ok)
{
    return kepler_warm_wide_finish<POLISH2>(e, K0, Mn, kepler_warm_pre(e, K0, Mn), ok);
}

// How far outside kepler_warm_wide's accuracy domain the step of prefix w is: acceptable when the
// returned ratio is <= 1 (its three tests; the quadratic one enters as a square root so that the ratio
// scales like 1/ns under ns equal sub-steps in M).
__device__ __forceinline__ float kepler_warm_need_pre(const WarmPre &w)
{
    const float lin = (float)fmax(w.ax * (1.0 / 0.3), w.axa2 * (1.0 / 0.08));
    const float cub = sqrtf((float)(fabs(w.ec * w.rg) * w.x * w.x * (1.0 / (6.0 * 0.02))));
    return fmaxf(lin, cub);
}

// Re-synchronise (sin E, cos E) with E = M + u exactly (libdevice sincos of the reduced angle), u
// untouched: the survivors of the cull start their polishes from here, so that neither the
// truncation of the cull-quality rotations nor their rounding can reach a refined pair.
__device__ __forceinline__ Kepler kepler_resync(const Kepler &K0)
{
    const double k = rint(K0.M * kInvTwoPi);
    double m = fma(-k, kTwoPiHi, K0.M);
    m = fma(-k, kTwoPiLo, m);
    Kepler K = K0;
    sincos(m + K0.u, &K.s, &K.c);
    return K;
}

// Refresh: recompute (sin E, cos E) of the carried state exactly (libdevice sincos of the reduced
// E = M + u) and polish u once, so the rounding of the Taylor rotations cannot accumulate beyond
// one exposure group.
__device__ __forceinline__ Kepler kepler_refresh(double e, const Kepler &K0)
{
    const double k = rint(K0.M * kInvTwoPi);
    double m = fma(-k, kTwoPiHi, K0.M);
    m = fma(-k, kTwoPiLo, m);
    double s, c;
    sincos(m + K0.u, &s, &c);
    const double f = fma(-e, s, K0.u);
    const double g = fma(-e, c, 1.0);
    const double d = -f * rcp_nr<2>(g);
    Kepler K;
    K.M = K0.M;
    K.u = K0.u + d;
    K.s = fma(d, c, s);
    K.c = fma(-d, s, c);
    return K;
}

// ---- group ephemeris gate (reading A25) ------------------------------------------------------------
// A blind search culls all but ~1e-6 of its pairs, and the cull above still pays a Kepler step per pair.  The gate
// replaces that step, for one exposure group at a time, by the second-order Taylor expansion of the heliocentric
// position about the group's mid-time tm,
//     T2(tau) = r + v tau + (a/2) tau^2,   v = (dE/dt)(-A sin E + B cos E),  dE/dt = n / (1 - e cos E),
//                                           a = -(GM / |r|^3) r = -n^2 (1 - e cos E)^-3 r,
// from ONE polished Kepler solve per (orbit, group), and culls a pair when T2 - R_obs lies outside a cone that is
// widened by everything T2 leaves out -- rigorously, so that no pair the exact path would report can be lost:
//   * Taylor remainder: |r(t) - T2| <= |tau|^3 / 6 sup |d3r/dt3|, and d3r/dt3 = -GM (v / r^3 - 3 (r.v) r / r^5)
//     gives |d3r/dt3| <= 4 GM |v| / r^3; over the group r >= rmin (below) and |v| <= min(vmax, sqrt(2 GM / rmin))
//     (vmax: perihelion speed), tau_max the group's half-span;
//   * light-time: |r(t - lt) - r(t)| <= vmax lt, lt = rho / c, rho <= D / cos(theta_c) <= D (1 + tan theta_c);
//   * footprint: a hit has D = q.t > 0 and a distance from the pointing axis d_perp <= D tan(theta_c), theta_c the
//     footprint's half-diagonal (tan_fov, exact for the gnomonic projection).
// With |delta| <= eps_tot the displacement between the true topocentric vector and T2 - R_obs, D0 and d0 the
// approximate vector's axial and perpendicular components: D0 >= D - eps_tot and d0 <= (D0 + eps_tot) tan(theta_c)
// + eps_tot, eps_tot <= (epsT + kappa D0)(1 + 2 kappa), kappa = vmax / (c cos theta_c).  The gate therefore keeps a
// pair unless D0 < -eps or d0 > D0 tq + eps, with tq and eps below (5 % margins on every term; comparisons are
// written so that a NaN keeps the pair).  Nothing else changes: a pair the gate keeps goes through the cull-quality
// chain and the exact cone test as before, from a Kepler state that is at most half a group old.
// The per-pair test runs in FP32 -- it is a filter with explicit margins, not a result -- so that it costs FP32-pipe
// issue slots instead of FP64 ones.  Its rounding enters the bound like everything else T2 leaves out.  With u = 2^-24:
//   * the FP32 vector p~ = fl(fl(fma(fl(fma(h~, tau~, v~)), tau~, r~)) - R~) from inputs rounded to FP32 differs from
//     T2 - R_obs by <= 6 u A per component, A = |r| + |v| tau_max + |a/2| tau_max^2 + max |R_obs| (three roundings of
//     the inputs and two of the operations on each term at most); 24 u A (2.3 x the vector norm of that) is added to
//     the displacement bound epsT, so p~ takes the place of T2 - R_obs in the derivation above;
//   * D~ = fl(p~ . t~) is off by <= 6 u |p~| and r2~ = fl(p~ . p~) by <= 3 u |p~|^2, hence fma(-D~, D~, r2~) differs
//     from |p~|^2 - (p~ . t)^2 by <= 16 u |p~|^2: the test compares it with w^2 + 40 u r2~, w = D~ tq + eps with tq
//     and eps rounded UP after a factor (1 + 32 u) that covers the roundings of w itself and of D~ inside it.
//     (On the far side, D~ < -eps can only be reached by vectors with |p~| <= 1.5 eps, where 6 u |p~| << 32 u eps.)
struct GroupEph {
    float rx, ry, rz, vx, vy, vz, hx, hy, hz;       // r, v, a / 2 at the expansion time tm: heliocentric equatorial
    float tq, eps;                                  // keep unless D0 < -eps or d0 > D0 tq + eps (+ rounding slack)
};
constexpr float kGateU = 5.9604645e-8f;             // 2^-24

// The gate's two constants.  rmin: a lower bound of |r| over the group.  MUFU seeds + one Newton / Goldschmidt step
// (1e-12 relative) are plenty under 5 % margins.
__device__ __forceinline__ double gate_eps_bound(double gm, double vmax, double rmin, double tau_max, double tan_fov)
{
    const double rinv = rcp_nr<1>(rmin);
    const double vint = fmin(vmax, sqrt_nr<1>(2.0 * gm * rinv));
    const double epsT = 1.05 * (4.0 * gm * vint * (rinv * rinv * rinv)) * (tau_max * tau_max * tau_max) * (1.0 / 6.0);
    return fma(1.05 * epsT, 1.0 + tan_fov, 1e-12);
}
__device__ __forceinline__ double gate_tq(double vmax, double inv_c, double tan_fov)
{
    const double kap = 1.05 * vmax * inv_c * (1.0 + tan_fov);   // >= vmax / (c cos theta_c), and its (1 + 2 kappa)
    // a light-time cone that is no cone (kappa >~ 0.01 needs e -> 1): infinite, the gate then keeps every pair
    return (kap < 0.01) ? fma(kap, 1.0 + tan_fov, 1.01 * tan_fov) + 1e-9 : INFINITY;
}

// K: the POLISHED Kepler state at tm.  a: semi-major axis.  tau_max: max |t_j - tm| over the group.  r_obs_max: an
// upper bound of the observer's heliocentric distance over the group.
__device__ __forceinline__ GroupEph group_ephemeris(const Orbit &o, double a, const Kepler &K, double tau_max,
                                                    double r_obs_max, double gm, double inv_c, double tan_fov)
{
    GroupEph G;
    const double g = fma(-o.e, K.c, 1.0);
    const double rg = rcp_nr<2>(g);
    const double X = K.c - o.e;
    G.rx = __double2float_rn(fma(o.Ax, X, o.Bx * K.s));
    G.ry = __double2float_rn(fma(o.Ay, X, o.By * K.s));
    G.rz = __double2float_rn(fma(o.Az, X, o.Bz * K.s));
    const double w = o.n * rg;                                   // dE/dt
    G.vx = __double2float_rn(w * fma(o.Bx, K.c, -o.Ax * K.s));
    G.vy = __double2float_rn(w * fma(o.By, K.c, -o.Ay * K.s));
    G.vz = __double2float_rn(w * fma(o.Bz, K.c, -o.Az * K.s));
    const double k = -0.5 * (o.n * o.n) * (rg * rg * rg);        // a / 2 = k r
    G.hx = __double2float_rn(k * fma(o.Ax, X, o.Bx * K.s));
    G.hy = __double2float_rn(k * fma(o.Ay, X, o.By * K.s));
    G.hz = __double2float_rn(k * fma(o.Az, X, o.Bz * K.s));
    const double r = a * g;
    const double tq = gate_tq(o.vmax, inv_c, tan_fov);
    // |r| over the group: no closer than the perihelion, no closer than |r(tm)| minus the longest way the object can go
    double eps = gate_eps_bound(gm, o.vmax, fmax(a * (1.0 - o.e), fma(-o.vmax, tau_max, r)), tau_max, tan_fov);
    // the FP32 evaluation of the vector (see above): |v| <= vmax, |a / 2| = -k r
    const double A = r + o.vmax * tau_max + (-k * r) * (tau_max * tau_max) + r_obs_max;
    eps = fma(24.0 * (double)kGateU * A, 1.0 + tan_fov, eps);
    if (!(tq < 1e30) || !(eps < 1e30)) eps = INFINITY;           // no cone, or anything non-finite: keep every pair
    G.tq = __double2float_ru(tq * (1.0 + 32.0 * (double)kGateU));
    G.eps = __double2float_ru(eps * (1.0 + 32.0 * (double)kGateU));
    return G;
}

// true: the pair cannot be a hit.  tau = t_exposure - tm, R the observer at the exposure, t the unit vector to its
// tangent point, all rounded to FP32.  A NaN keeps the pair.
__device__ __forceinline__ bool group_gate_culls(const GroupEph &G, float tau, float Rx, float Ry, float Rz, float tx,
                                                 float ty, float tz)
{
    const float px = fmaf(fmaf(G.hx, tau, G.vx), tau, G.rx) - Rx;
    const float py = fmaf(fmaf(G.hy, tau, G.vy), tau, G.ry) - Ry;
    const float pz = fmaf(fmaf(G.hz, tau, G.vz), tau, G.rz) - Rz;
    const float r2 = fmaf(px, px, fmaf(py, py, pz * pz));
    const float D0 = fmaf(px, tx, fmaf(py, ty, pz * tz));
    const float w = fmaf(D0, G.tq, G.eps);
    return (D0 < -G.eps) || (fmaf(-D0, D0, r2) > fmaf(w, w, 40.0f * kGateU * r2));
}

// ---- group-level test: can the orbit be near ANY exposure of the group? ---------------------------------------------
// Where a group's pointings cluster (a survey that follows the opposition point), most orbits are nowhere near any of its
// 32 exposures, and one test per (orbit, group) replaces 32.  Per group (k_group_bounds, once per launch): the axis c of the
// pointings, alpha = 1.01 theta_c + max_j angle(t_j, c) + 1e-4, the mean observer position R_m and dR = max_j |R_j - R_m|.
// The retarded topocentric vector of exposure j is p_j = [r(t_m) - R_m] + [r(t_j - lt) - r(t_m)] - [R_j - R_m], i.e. within
// rho_b = v_max (tau_max + lt) + dR of p_m = r(t_m) - R_m (speed bound; lt <= (|p_m| + rho_b) / c), so its direction is within
// asin(rho_b / |p_m|) of p_m's, and a hit needs angle(p_j, t_j) <= theta_c.  Hence no exposure of the group can be hit when
//     angle(p_m, c) > alpha + asin(rho_b / |p_m|) =: Theta   (Theta < pi / 2),
// tested as p_m . c < |p_m| cos(Theta) with cos(Theta) = cos(alpha) sqrt(1 - s^2) - sin(alpha) s, s = rho_b / |p_m| < 1.
// FP32 with margins: 1e-4 AU on rho_b for the rounding of p_m (<= 1e-5 AU at 50 AU), 1e-5 relative and 1e-6 AU absolute on
// the comparison.  bounds: (c, cos alpha), (R_m, dR), (sin alpha, -, -, -); cos alpha = -2 marks a group without a usable cone.
__device__ __forceinline__ bool group_is_far(float rx, float ry, float rz, float vmax, float tau_max, float inv_c,
                                             float4 b0, float4 b1, float4 b2)
{
    const float px = rx - b1.x, py = ry - b1.y, pz = rz - b1.z;
    const float pm2 = fmaf(px, px, fmaf(py, py, pz * pz));
    const float pm = sqrtf(pm2);
    float rho_b = fmaf(vmax, tau_max, b1.w) + 1e-4f;
    rho_b = fmaf(1.05f * vmax * inv_c, pm + 2.f * rho_b, rho_b);        // light-time: v_max (|p_m| + rho_b) / c, with room
    const float s = rho_b / pm;
    const float cosT = fmaf(b0.w, sqrtf(fmaxf(1.f - s * s, 0.f)), -b2.x * s);
    const float pc = fmaf(px, b0.x, fmaf(py, b0.y, pz * b0.z));
    // written so that a NaN anywhere means "not far"
    return (s < 0.98f) && (b0.w > -1.f) && (cosT > 1e-3f) && (pc < fmaf(pm, cosT * (1.f - 1e-5f), -1e-6f));
}

}  // namespace dt
