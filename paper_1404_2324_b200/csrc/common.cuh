// Device-side building blocks shared by all kernels of the hybrid symplectic step.
// Citations are to PAPER.md (Grimm & Stadel, GENGA) lines / equations.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace genga {

// error bits latched in the device status word
enum : int { ERRBIT_CAPACITY = 1, ERRBIT_KEPLER = 2, ERRBIT_BS = 4 };

// device counters (int64 slots in DevCounters::c)
enum : int { CNT_GROUPS = 0, CNT_MAXGROUP = 1, CNT_BSSTEPS = 2, CNT_CAND = 3, CNT_BSREJECTS = 4, CNT_NEV = 5, CNT_STEPID = 6, CNT_N = 8 };

// ---------------------------------------------------------------------------------
// Changeover function K (Eq. 4-5) and the weight of the Newtonian pair force
// in the kick, W = K - r dK/dr: the exact gradient of H_B (Eq. 2 L76 through Eq. 8).
// The direct part H_A (Eq. 1) carries 1 - W.
__device__ __forceinline__ double kick_weight(double r, double rc)
{
    double y = (r - 0.1 * rc) / (0.9 * rc);
    if (!(y > 0.0)) return 0.0;          // also rc == 0 && r == 0
    if (y >= 1.0) return 1.0;
    double D = 2.0 * y * y - 2.0 * y + 1.0;
    double K = y * y / D;
    double dK = 2.0 * y * (1.0 - y) / (D * D) / (0.9 * rc);
    return K - r * dK;
}

// ---------------------------------------------------------------------------------
// FP64 reciprocal square root, x^(-3/2) and reciprocal from the hardware seeds MUFU.RSQ64H /
// MUFU.RCP64H (relative error <= 2^-19, measured) plus ONE third-order correction step in
// DFMA arithmetic.  For positive normal x.  Measured over 1.5e8 samples on B200 (DESIGN.md
// "Arithmetic"): rsqrt_fast max 1.25 ulp, rinv3_fast <= ~4 ulp, rcp_fast 0.51 ulp, all with
// mean signed error < 0.005 ulp (unbiased).  The paper keeps IEEE sqrt and divide for fear
// of a *biased* rsqrt (L228, L264); these are unbiased and far inside the 1e-12 parity bound,
// and they cost 5-7 FP64 issue slots instead of the ~25 of sqrt followed by a divide.
__device__ __forceinline__ double rsqrt_seed(double x) { double y; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); return y; }
__device__ __forceinline__ double rcp_seed(double x) { double y; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); return y; }
__device__ __forceinline__ double rsqrt_fast(double x)
{
    double y0 = rsqrt_seed(x);
    double e = fma(-x * y0, y0, 1.0);              // 1 - x y0^2
    double p = fma(0.375, e, 0.5);
    return fma(p * e, y0, y0);                     // y0 (1 + e/2 + 3 e^2/8)
}
__device__ __forceinline__ double rinv3_fast(double x)   // x^(-3/2)
{
    double y0 = rsqrt_seed(x);
    double u = y0 * y0;
    double e = fma(-x, u, 1.0);
    double w = y0 * u;
    double p = fma(1.875, e, 1.5);
    return fma(p * e, w, w);                       // y0^3 (1 + 3e/2 + 15 e^2/8)
}
__device__ __forceinline__ double rcp_fast(double x)
{
    double r0 = rcp_seed(x);
    double e = fma(-x, r0, 1.0);
    return fma(r0, fma(e, e, e), r0);              // r0 (1 + e + e^2)
}

// Weight of the Newtonian pair force that stays in H_A (Eq. 1), times G m_j / d^3, for a
// pair inside the changeover zone (d2 < rc_ij^2): G m_j (1 - W(d, rc_ij)) / d^3.  Same function
// as 1 - kick_weight(), arranged without sqrt or divide (irc09 = 1 / (0.9 rc_ij)) because
// Bulirsch-Stoer evaluates it on a latency-bound dependent chain.
__device__ __forceinline__ double direct_scale(double d2, double rcij, double irc09, double Gmj)
{
    // 1 - W = 1 - K + r dK/dr = [D^2 - y^2 D + 2 r y (1 - y) / (0.9 rc)] / D^2,  D = 2 y^2 - 2 y + 1:
    // one reciprocal (of D^2) at the end of the chain, the numerator is ready before it
    // d and 1/d from the same seed, d without the extra multiply at the end of the chain
    const double y0 = rsqrt_seed(d2), t0 = d2 * y0;
    const double e0 = fma(-t0, y0, 1.0);
    const double pe = fma(0.375, e0, 0.5) * e0;
    double dd = fma(pe, t0, t0);                                  // d2 y0 (1 + e/2 + 3 e^2/8) = sqrt(d2)
    double rinv = fma(pe, y0, y0);
    double y = (dd - 0.1 * rcij) * irc09;
    double w1 = 1.0;
    if (y > 0.0) {
        double D = fma(2.0 * y, y - 1.0, 1.0);
        double N = fma(D, D - y * y, 2.0 * (dd * irc09) * (y * (1.0 - y)));
        w1 = N * rcp_fast(D * D);
    }
    return Gmj * (rinv * rinv) * rinv * w1;
}

// G m_j (1 - W(d, rc_ij)) / d^3 as direct_scale(), without a branch (all lanes of a warp run it
// together; `in` selects afterwards).
__device__ __forceinline__ double direct_scale_nb(double d2, double rcij, double irc09, double Gmj)
{
    // d and 1/d from the same seed, d without the extra multiply at the end of the chain
    const double y0 = rsqrt_seed(d2), t0 = d2 * y0;
    const double e0 = fma(-t0, y0, 1.0);
    const double pe = fma(0.375, e0, 0.5) * e0;
    double dd = fma(pe, t0, t0);                                  // d2 y0 (1 + e/2 + 3 e^2/8) = sqrt(d2)
    double rinv = fma(pe, y0, y0);
    double y = (dd - 0.1 * rcij) * irc09;
    double D = fma(2.0 * y, y - 1.0, 1.0);                    // >= 1/2 for every y
    double N = fma(D, D - y * y, 2.0 * (dd * irc09) * (y * (1.0 - y)));
    double w1 = N * rcp_fast(D * D);
    w1 = y > 0.0 ? w1 : 1.0;
    return Gmj * (rinv * rinv) * rinv * w1;
}

// ---------------------------------------------------------------------------------
// Stumpff functions c0..c3 at x (Danby 1988; named at L110, L230).  Bounded work:
// argument quartering down to |x| <= 1 (at most 20 times), degree-9 series, then the
// quadruple-angle recurrences.
__device__ __forceinline__ void stumpff(double x, double &c0, double &c1, double &c2, double &c3)
{
    int n = 0;
    while (fabs(x) > 1.0 && n < 20) { x *= 0.25; ++n; }
    // c2 = sum (-x)^k/(2k+2)!, c3 = sum (-x)^k/(2k+3)!
    double z = -x;
    double a2 = 1.0 / 6402373705728000.0;            // 1/18!
    a2 = fma(a2, z, 1.0 / 20922789888000.0);         // 1/16!
    a2 = fma(a2, z, 1.0 / 87178291200.0);            // 1/14!
    a2 = fma(a2, z, 1.0 / 479001600.0);              // 1/12!
    a2 = fma(a2, z, 1.0 / 3628800.0);                // 1/10!
    a2 = fma(a2, z, 1.0 / 40320.0);                  // 1/8!
    a2 = fma(a2, z, 1.0 / 720.0);                    // 1/6!
    a2 = fma(a2, z, 1.0 / 24.0);                     // 1/4!
    a2 = fma(a2, z, 0.5);                            // 1/2!
    double a3 = 1.0 / 121645100408832000.0;          // 1/19!
    a3 = fma(a3, z, 1.0 / 355687428096000.0);        // 1/17!
    a3 = fma(a3, z, 1.0 / 1307674368000.0);          // 1/15!
    a3 = fma(a3, z, 1.0 / 6227020800.0);             // 1/13!
    a3 = fma(a3, z, 1.0 / 39916800.0);               // 1/11!
    a3 = fma(a3, z, 1.0 / 362880.0);                 // 1/9!
    a3 = fma(a3, z, 1.0 / 5040.0);                   // 1/7!
    a3 = fma(a3, z, 1.0 / 120.0);                    // 1/5!
    a3 = fma(a3, z, 1.0 / 6.0);                      // 1/3!
    c2 = a2; c3 = a3;
    c1 = fma(z, c3, 1.0);
    c0 = fma(z, c2, 1.0);
    for (; n > 0; --n) {
        c3 = 0.25 * (c2 + c0 * c3);
        c2 = 0.5 * c1 * c1;
        c1 = c0 * c1;
        c0 = 2.0 * c0 * c0 - 1.0;
    }
}

// Kepler drift of one body about mu = G m0 (L114) for time h by Gauss' f and g functions
// (Eq. 9) in universal variables (L230).  Solve
//   F(s) = r0 s c1 + u s^2 c2 + mu s^3 c3 - h = 0,  c_k at alpha s^2,
// with a bounded quartic-convergence Newton iteration (F' = r, F'' , F''' closed form);
// if that has not converged in KEPLER_MAXIT steps, fall back to bracketed bisection/Newton.
// Returns false if neither converged (caller latches ERRBIT_KEPLER).
constexpr int KEPLER_MAXIT = 10;

static __device__ __noinline__ bool kepler_solve_slow(double mu, double h, double r0, double u, double alpha, double &s_out)
{
    double s = h / r0, lo = -INFINITY, hi = INFINITY;
    for (int it = 0; it < 80; ++it) {
        double c0, c1, c2, c3;
        stumpff(alpha * s * s, c0, c1, c2, c3);
        double F = r0 * s * c1 + u * s * s * c2 + mu * s * s * s * c3 - h;
        double r = r0 * c0 + u * s * c1 + mu * s * s * c2;
        if (F > 0.0) { if (s < hi) hi = s; } else if (F < 0.0) { if (s > lo) lo = s; }
        double sn = s - F / r;
        if (!(sn > lo && sn < hi)) {
            if (isfinite(lo) && isfinite(hi)) sn = 0.5 * (lo + hi);
            else if (!isfinite(sn)) return false;
        }
        double step = fabs(sn - s);
        s = sn;
        if (step <= 1e-15 * fabs(s)) { s_out = s; return true; }
    }
    return false;
}

__device__ __forceinline__ bool kepler_drift(double mu, double h, double &x, double &y, double &z,
                                             double &vx, double &vy, double &vz)
{
    // reciprocals by rcp_fast / rsqrt_fast (0.5 / 1.25 ulp, above): an IEEE divide or square root costs
    // 14-20 FP64 issue slots and the particle pass is bound by them
    double r02 = x * x + y * y + z * z;
    double ir0 = rsqrt_fast(r02);
    double r0 = r02 * ir0;
    double v2 = vx * vx + vy * vy + vz * vz;
    double u = x * vx + y * vy + z * vz;
    double alpha = 2.0 * mu * ir0 - v2;
    double k3 = mu - alpha * r0;
    double s = h * ir0;
    double G0, G1, G2, G3, r;                                 // G_k = s^k c_k(alpha s^2)
    bool ok = false;
#pragma unroll 1
    for (int it = 0; it < KEPLER_MAXIT; ++it) {
        double c1, c2, c3;
        stumpff(alpha * s * s, G0, c1, c2, c3);
        G1 = s * c1; G2 = s * s * c2; G3 = s * s * s * c3;
        double F = r0 * G1 + u * G2 + mu * G3 - h;
        r = r0 * G0 + u * G1 + mu * G2;                       // dF/ds
        double F2 = k3 * G1 + u * G0;                         // second derivative
        double F3 = k3 * G0 - alpha * u * G1;                 // third derivative
        double d = -F * rcp_fast(r);
        d = -F * rcp_fast(r + 0.5 * d * F2);
        d = -F * rcp_fast(r + 0.5 * d * F2 + d * d * F3 * (1.0 / 6.0));
        if (fabs(d) <= 1e-6 * fabs(s) && fabs(F) <= 1e-5 * fabs(h)) {   // in the basin: quartic convergence
            // the last correction: carried into the G functions by their Taylor series (dG0 = -alpha G1,
            // dG1 = G0, dG2 = G1, dG3 = G2), truncation O(d^3) < 1e-18 relative: saves the confirming pass
            const double hd2 = 0.5 * d * d;
            const double n0 = G0 - alpha * (G1 * d + G0 * hd2);
            const double n1 = G1 + G0 * d - alpha * G1 * hd2;
            const double n2 = G2 + G1 * d + G0 * hd2;
            const double n3 = G3 + G2 * d + G1 * hd2;
            G0 = n0; G1 = n1; G2 = n2; G3 = n3;
            r = r0 * G0 + u * G1 + mu * G2;
            ok = true;
            break;
        }
        s += d;
    }
    if (!ok) {
        if (!kepler_solve_slow(mu, h, r0, u, alpha, s)) return false;
        double c1, c2, c3;
        stumpff(alpha * s * s, G0, c1, c2, c3);
        G1 = s * c1; G2 = s * s * c2; G3 = s * s * s * c3;
        r = r0 * G0 + u * G1 + mu * G2;
    }
    double ir = rcp_fast(r);
    double f = 1.0 - mu * G2 * ir0;
    double g = h - mu * G3;
    double fd = -mu * G1 * (ir * ir0);
    double gd = 1.0 - mu * G2 * ir;
    double nx = f * x + g * vx, ny = f * y + g * vy, nz = f * z + g * vz;
    double nvx = fd * x + gd * vx, nvy = fd * y + gd * vy, nvz = fd * z + gd * vz;
    x = nx; y = ny; z = nz; vx = nvx; vy = nvy; vz = nvz;
    return true;
}

// ---------------------------------------------------------------------------------
// Minimum over the drift of the cubic Hermite interpolant of the squared separation
// (Eq. 10-12).  P = |dq|^2, Pd = 2 dq.dV at both ends; dP/dt = a t^2 + b t + c with
// a = 6(P0-P1) + 3h(Pd0+Pd1)  [the minus printed at L128 contradicts Eq. 10], b, c as printed.
__device__ __forceinline__ double hermite_P(double t, double P0, double P1, double Pd0, double Pd1, double h)
{
    double o = 1.0 - t;
    return o * o * (1.0 + 2.0 * t) * P0 + t * t * (3.0 - 2.0 * t) * P1 + t * o * o * h * Pd0 - t * t * o * h * Pd1;
}
__device__ __forceinline__ double hermite_min(double P0, double P1, double Pd0, double Pd1, double h)
{
    double a = 6.0 * (P0 - P1) + 3.0 * h * (Pd0 + Pd1);
    double b = 6.0 * (P1 - P0) - 2.0 * h * (2.0 * Pd0 + Pd1);
    double c = h * Pd0;
    double D = fmin(P0, P1);
    double t0 = -1.0, t1 = -1.0;
    if (a == 0.0) { if (b != 0.0) t0 = -c / b; }
    else {
        double disc = b * b - 4.0 * a * c;
        if (disc >= 0.0) {
            double sq = sqrt(disc);
            double qq = -0.5 * (b + (b >= 0.0 ? sq : -sq));
            t0 = qq / a;
            if (qq != 0.0) t1 = c / qq;
        }
    }
    if (t0 > 0.0 && t0 < 1.0) D = fmin(D, hermite_P(t0, P0, P1, Pd0, Pd1, h));
    if (t1 > 0.0 && t1 < 1.0) D = fmin(D, hermite_P(t1, P0, P1, Pd0, Pd1, h));
    return D;
}

// Yoshida (1990) substep weights (L168-170); order 6 = "solutions A".
__host__ __device__ inline int yoshida_weights(int order, double w[7])
{
    if (order == 2) { w[0] = 1.0; return 1; }
    if (order == 4) {
        const double cbrt2 = 1.2599210498948731648;
        double w1 = 1.0 / (2.0 - cbrt2);
        w[0] = w1; w[1] = 1.0 - 2.0 * w1; w[2] = w1;
        return 3;
    }
    if (order == 6) {
        const double a1 = -1.17767998417887, a2 = 0.235573213359357, a3 = 0.784513610477560;
        const double a0 = 1.0 - 2.0 * (a1 + a2 + a3);
        w[0] = a3; w[1] = a2; w[2] = a1; w[3] = a0; w[4] = a1; w[5] = a2; w[6] = a3;
        return 7;
    }
    return 0;
}

}  // namespace genga
