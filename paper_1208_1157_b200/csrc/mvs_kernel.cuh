// mvs_kernel.cuh — the fused mixed-variable-symplectic step loop for sm_100a (FP64 CUDA cores).
//
// One launch = Alg. 1 for every system with the MVS propagator of P:L99-125 / P:L254-256 in
// democratic-heliocentric variables (reading R-M1: heliocentric positions Q_i = x_i - x_0, barycentric velocities
// V_i = v_i - V_cm, centre of mass X_cm, V_cm).  The state is converted once at load, lives in registers for all
// steps, and is converted back once at store.  One step (five sub-steps, kept unmerged, R-M7):
//   1  Q_i += h/2 s,  s = sum_k m_k V_k / m_0;  X_cm += h/2 V_cm          Cartesian drift
//   2  V_i += h/2 A_i                                                     kick, planets only
//   3  (Q_i, V_i) <- Kepler flow about mu = G m_0 for h                   Kepler drift             (R-M2)
//   4  A = planet-planet accelerations at the new Q, each pair once       (reused by step k+1's sub-step 2,
//      V_i += h/2 A_i                                                      P:L256)
//   5  Q_i += h/2 s (s from the new V; the SAME s opens the next step), X_cm += h/2 V_cm
// The Kepler drift uses universal variables (BASELINE.json config 4; R-M3, R-M4): solve
//   r0 G1 + eta G2 + mu G3 = tau,  G_n = X^n c_n(beta X^2),  then the f and g functions (kepler_drift_all: a straight-line
// fast path for steps of a few per cent of a period, the general procedure out of line).
//
// Work split: L lanes per system (L odd), B planets per lane; the Kepler drift is per planet and needs no
// communication; planet-planet pairs use the same in-lane + lane-ring schedule as the Hermite kernel (acc_pairs.cuh); the
// momentum sum of the Cartesian drift is an L-lane all-gather of per-lane partial sums.  L = 1 (n_body <= 9) is
// one system per thread with the oracle's summation order and no shuffle.  Monitors and loop tests: one quick test per
// step on high words and one vote, the exact logic behind a warp-uniform, rarely taken branch (as in hermite_kernel.cuh).
#pragma once
#include <cfloat>
#include <type_traits>

#include "acc_pairs.cuh"

namespace ensd {

// Stumpff functions c_n(z) = sum_k (-z)^k / (2k+n)!  (R-M3), series part: valid for |z| <= 0.1 (7 terms: truncation
// < 1e-20 relative).  For the step sizes of the workloads (h << orbital period) z = beta X^2 is always in this range.
__constant__ double kStumpff[16] = {
    // descending powers of z, c2 / c3 interleaved: -1/16!, -1/17!, 1/14!, 1/15!, ..., 1/2!, 1/3!
    -1.0 / 20922789888000.0, -1.0 / 355687428096000.0, 1.0 / 87178291200.0, 1.0 / 1307674368000.0,
    -1.0 / 479001600.0,      -1.0 / 6227020800.0,      1.0 / 3628800.0,     1.0 / 39916800.0,
    -1.0 / 40320.0,          -1.0 / 362880.0,          1.0 / 720.0,         1.0 / 5040.0,
    -1.0 / 24.0,             -1.0 / 120.0,             0.5,                 1.0 / 6.0};

__device__ __forceinline__ void stumpff_series(double z, double& c0, double& c1, double& c2, double& c3) {
    // Horner in z; the coefficients are constant-bank operands of the DFMAs (no registers, no immediates to build)
    // Seven terms (up to z^6): for |z| <= 0.1 the z^7 terms are < 5e-21 of c2 = 1/2, c3 = 1/6.  The leading (z^6)
    // coefficients 1/14!, 1/15! are literals truncated to their high words (their terms are < 1.2e-17, the truncation
    // error < 6e-24): built with one move each, so that the first DFMA does not wait for a constant load (a DFMA takes
    // one constant-bank operand).
    double s2 = 0x1.93974p-37, s3 = 0x1.ae7f3p-41;
#pragma unroll
    for (int k = 2; k < 8; ++k) {
        s2 = fma(s2, z, kStumpff[2 * k]);
        s3 = fma(s3, z, kStumpff[2 * k + 1]);
    }
    c2 = s2;
    c3 = s3;
    c1 = fma(-z, c3, 1.0);
    c0 = fma(-z, c2, 1.0);
}

struct Stumpff {
    double c0, c1, c2, c3;
};

// General argument: |z| is quartered until <= 0.1, the series is summed there, and c_n(4z) is rebuilt from c_n(z) by
// the duplication formulas.  Out of line (returns in registers): only steps of a sizeable fraction of an orbital
// period come here.
__device__ __noinline__ Stumpff stumpff_general(double z) {
    int nq = 0;
    // at most 540 quarterings bring any finite double below 0.1; +-inf and NaN leave the loop at the bound and give
    // non-finite G functions, which the non-finite monitor reports (no endless loop on a broken state)
    while (fabs(z) > 0.1 && nq < 540) {
        z *= 0.25;
        ++nq;
    }
    if (!(fabs(z) <= 0.1)) z = __longlong_as_double(0x7ff8000000000000ll);
    Stumpff c;
    stumpff_series(z, c.c0, c.c1, c.c2, c.c3);
    for (; nq > 0; --nq) {
        const double n3 = 0.25 * fma(c.c0, c.c3, c.c2);
        const double n2 = 0.5 * c.c1 * c.c1;
        const double n1 = c.c0 * c.c1;
        const double n0 = fma(2.0 * c.c0, c.c0, -1.0);
        c.c3 = n3;
        c.c2 = n2;
        c.c1 = n1;
        c.c0 = n0;
    }
    return c;
}

struct KeplerG {
    double G0, G1, G2, G3;
};

__device__ __forceinline__ KeplerG kepler_G_from(const Stumpff& c, double X, double X2) {
    KeplerG g;
    g.G0 = c.c0;
    g.G1 = X * c.c1;
    g.G2 = X2 * c.c2;
    g.G3 = (X2 * X) * c.c3;
    return g;
}

__device__ __forceinline__ KeplerG kepler_G(double beta, double X) {  // general argument (fallback path only)
    const double X2 = X * X;
    return kepler_G_from(stumpff_general(beta * X2), X, X2);
}

// Residual of the universal Kepler equation; monotone in X (its derivative is the radius r > 0).
__device__ __forceinline__ double kepler_resid(double r0, double eta, double mu, double beta, double tau, double X) {
    const KeplerG g = kepler_G(beta, X);
    return fma(r0, g.G1, fma(eta, g.G2, fma(mu, g.G3, -tau)));
}

// Guaranteed-convergent fallback (R-M4): bracket the root and bisect.  Out of line: essentially never taken.
__device__ __noinline__ double kepler_bisect(double r0, double eta, double mu, double beta, double tau) {
    double lo = 0.0, hi = tau / r0;
    const double sgn = tau >= 0.0 ? 1.0 : -1.0;
    if (hi == 0.0) hi = sgn;
    for (int k = 0; k < 200 && sgn * kepler_resid(r0, eta, mu, beta, tau, hi) < 0.0; ++k) hi *= 2.0;
    for (int k = 0; k < 200; ++k) {
        const double mid = 0.5 * (lo + hi);
        if (sgn * kepler_resid(r0, eta, mu, beta, tau, mid) < 0.0)
            lo = mid;
        else
            hi = mid;
    }
    return 0.5 * (lo + hi);
}

// |x| as the high word of its bit pattern (sign cleared): exponent and the top 20 mantissa bits.  Order-preserving
// for finite values, NaN and inf sort at or above 0x7ff00000: threshold tests on the integer ALU instead of DSETP.
__device__ __forceinline__ int abs_hi(double x) { return __double2hiint(x) & 0x7fffffff; }
constexpr int kHi0p1 = 0x3fb99999;  // high word of 0.1 (0x3FB999999999999A), rounded down
constexpr int kHiInf = 0x7ff00000;
// a Chebyshev step below 2^-18 |X| leaves an error of order |dX / X|^3 < 2e-17: converged
constexpr double kConv = 3.814697265625e-06;
constexpr int kHiConv2 = 0x3db00000;  // high word of kConv^2 = 2^-36

// Kepler drift of the B planets of this lane about a fixed centre of gravitational parameter mu for time tau
// (R-M3, R-M4).  The same root as the oracle's plain Newton iteration, reached with fewer evaluations of
// the G functions, no IEEE divide, and straight-line code over the planets:
//   * the B planets are iterated together, every stage written as a loop over b with no branch inside, so that B
//     independent dependency chains are in flight (DFMA latency 8 cycles against an issue interval of 2: one Kepler
//     solve alone leaves the FP64 pipe mostly idle);
//   * each iteration is Newton's step d1 = F / F' with Chebyshev's third-order correction d1 (1 + F F'' / (2 F'^2)),
//     F' = r, F'' = eta G0 + (mu - beta r0) G1 (derivatives of the G functions: G0' = -beta G1, G_n' = G_{n-1});
//     the correction is dropped when it is not small, which leaves Newton's step;
//   * the iteration starts from the fourth-order series solution of the equation (below), not from X = tau / r0;
//   * when every planet's step is below 2^-18 |X| the iteration has converged to far below rounding (the error after
//     the step is of order |dX / X|^3), and the G functions at the final X follow from a second-order Taylor update
//     with those same derivatives (neglected terms < 1e-18 relative) instead of one more Stumpff evaluation;
//   * 1 / r0 comes from the reciprocal square root of |q|^2 and 1 / r from rcp_f64;
//   * Stumpff arguments beyond the series range (|z| > 0.1: steps of a sizeable fraction of a period) and lanes
//     that fail to converge within the cap take out-of-line general paths.
// valid(b) = false leaves slot b untouched (massless dummy slots of padded shapes).
// Fourth-order series start of the universal Kepler equation (see kepler_drift_all); returns the correction `corr`
// with X = u (1 + corr).
__device__ __forceinline__ double kepler_series_start(double u, double ir0, double r0, double eta, double beta, double mu) {
    const double e1 = eta * ir0, e2 = e1 * e1, br = beta * r0;
    const double k = mu - br;
    const double q3 = fma(-1.0 / 6.0, k * ir0, 0.5 * e2);
    const double q4 = fma(-0.625, e2 * e1, (e1 * ir0) * fma(1.0 / 24.0, br, (5.0 / 12.0) * k));
    return u * fma(u, fma(u, q4, q3), -0.5 * e1);
}

// The general procedure of the Kepler drift (R-M4), for the lanes the fast path of kepler_drift_all does not stand for:
// all B planets of the lane from the start.  Out of line (the state goes through local memory): rarely called.
template <int B>
struct KeplerLane {
    double r0[B], ir0[B], eta[B], beta[B], X[B], d[B];
    KeplerG g[B];
};
template <int B>
__device__ __noinline__ void kepler_general_solve(KeplerLane<B>& s, double mu, double tau) {
    double(&r0)[B] = s.r0;
    double(&ir0)[B] = s.ir0;
    double(&eta)[B] = s.eta;
    double(&beta)[B] = s.beta;
    double(&X)[B] = s.X;
    double(&d)[B] = s.d;
    KeplerG(&g)[B] = s.g;
    int ok[B];
#pragma unroll
    for (int b = 0; b < B; ++b) {
        const double u = tau * ir0[b];
        const double corr = kepler_series_start(u, ir0[b], r0[b], eta[b], beta[b], mu);
        X[b] = abs_hi(corr) < 0x3fd00000 ? fma(u, corr, u) : u;  // |corr| < 0.25
    }
    auto iterate = [&]() -> bool {
        double X2[B], z[B];
        Stumpff cs[B];
        int zmax = 0;
#pragma unroll
        for (int b = 0; b < B; ++b) {
            X2[b] = X[b] * X[b];
            z[b] = beta[b] * X2[b];
            zmax = max(zmax, abs_hi(z[b]));
        }
        if (zmax < kHi0p1) {
#pragma unroll
            for (int b = 0; b < B; ++b) stumpff_series(z[b], cs[b].c0, cs[b].c1, cs[b].c2, cs[b].c3);
        } else {
#pragma unroll
            for (int b = 0; b < B; ++b) cs[b] = stumpff_general(z[b]);
        }
        int conv = 1;
#pragma unroll
        for (int b = 0; b < B; ++b) {
            g[b] = kepler_G_from(cs[b], X[b], X2[b]);
            const double F = fma(r0[b], g[b].G1, fma(eta[b], g[b].G2, fma(mu, g[b].G3, -tau)));
            const double r = fma(r0[b], g[b].G0, fma(eta[b], g[b].G1, mu * g[b].G2));
            const double F2 = fma(eta[b], g[b].G0, fma(-beta[b], r0[b], mu) * g[b].G1);
            const double ir = rcp_f64<false>(r);
            const double d1 = F * ir;
            double c = (0.5 * d1) * (F2 * ir);
            c = abs_hi(c) < kHi0p1 ? c : 0.0;
            const double dX = fma(d1, c, d1);
            X[b] -= dX;
            d[b] = -dX;
            // converged when the step is small relative to X AND as an angle (beta dX^2 = the square of the step in
            // eccentric anomaly): the error left by a Chebyshev step is of the order of the cube of that angle,
            // which for steps of many revolutions (X large) is not small just because dX / X is
            ok[b] = (abs_hi(dX) <= abs_hi(kConv * X[b])) & (abs_hi((beta[b] * dX) * dX) <= kHiConv2) &
                    (abs_hi(X[b]) < kHiInf);
            conv &= ok[b];
        }
        return conv != 0;
    };
    bool done = iterate();
    for (int it = 1; it < 50 && !done; ++it) done = iterate();
    if (!done) {  // some planet of this lane did not converge within the cap (or went non-finite): bisect those
#pragma unroll
        for (int b = 0; b < B; ++b) {
            if (!ok[b]) {
                X[b] = kepler_bisect(r0[b], eta[b], mu, beta[b], tau);
                g[b] = kepler_G(beta[b], X[b]);
                d[b] = 0.0;
            }
        }
    }
}

template <int B, class Valid>
__device__ __forceinline__ void kepler_drift_all(double (&Q)[B][3], double (&P)[B][3], double mu, double tau,
                                                 unsigned amask, Valid valid) {
    double r0[B], ir0[B], eta[B], beta[B], X[B], d[B];
    KeplerG g[B];
    // The common case -- a step of a few per cent of a period -- is straight-line code with every test folded into one
    // flag (high words, integer ALU) and one vote: series start, ONE Stumpff series evaluation, one Chebyshev step.  It
    // stands when, for every planet of the lane, the start's correction is below 0.25, the Stumpff argument and the
    // Chebyshev correction are below 0.1, and the step taken is below 2^-18 |X| (with |z| < 0.1 that also bounds the
    // step as an angle: beta dX^2 < 0.1 * 2^-36).  Otherwise the lane redoes its planets with the general procedure
    // (kepler_general_solve: the same start and first iteration with their branches, then as many more as needed).
    // Where the fast path stands it has computed exactly what the general procedure computes: same results, bit for bit.
    int hcorr = 0, hz = 0, hc = 0, hX = 0, t1 = -0x7fffffff;
#pragma unroll
    for (int b = 0; b < B; ++b) {
        const double r02 = fma(Q[b][2], Q[b][2], fma(Q[b][1], Q[b][1], Q[b][0] * Q[b][0]));
        eta[b] = fma(Q[b][2], P[b][2], fma(Q[b][1], P[b][1], Q[b][0] * P[b][0]));
        const double v2 = fma(P[b][2], P[b][2], fma(P[b][1], P[b][1], P[b][0] * P[b][0]));
        ir0[b] = rsqrt_f64(r02);
        r0[b] = r02 * ir0[b];
        beta[b] = fma(2.0 * mu, ir0[b], -v2);
        // Starting value: the universal Kepler equation is the power series
        //   tau = r0 X + eta X^2 / 2 + (mu - beta r0) X^3 / 6 - beta eta X^4 / 24 + ...
        // and its reversion to fourth order in u = tau / r0,
        //   X = u (1 + u (q2 + u (q3 + u q4))),   q2 = -e1 / 2,  q3 = e1^2 / 2 - k / (6 r0),
        //   q4 = e1 (5 k / 12 + beta r0 / 24) / r0 - 5 e1^3 / 8,   e1 = eta / r0,  k = mu - beta r0,
        // is within 1e-6 of the root for steps of a few per cent of a period (config 4: max 7e-7), so that ONE
        // Chebyshev step reaches rounding level; the plain guess X = u (the oracle's, R-M4) needs two.  Same root.
        // Steps too long for the series (correction not small) start from X = u (kepler_general_solve).
        const double u = tau * ir0[b];
        const double corr = kepler_series_start(u, ir0[b], r0[b], eta[b], beta[b], mu);
        X[b] = fma(u, corr, u);
        hcorr = max(hcorr, abs_hi(corr));
    }
    {
        double X2[B], z[B];
        Stumpff cs[B];
#pragma unroll
        for (int b = 0; b < B; ++b) {
            X2[b] = X[b] * X[b];
            z[b] = beta[b] * X2[b];
            hz = max(hz, abs_hi(z[b]));
            stumpff_series(z[b], cs[b].c0, cs[b].c1, cs[b].c2, cs[b].c3);
        }
#pragma unroll
        for (int b = 0; b < B; ++b) {
            g[b] = kepler_G_from(cs[b], X[b], X2[b]);
            const double F = fma(r0[b], g[b].G1, fma(eta[b], g[b].G2, fma(mu, g[b].G3, -tau)));
            const double r = fma(r0[b], g[b].G0, fma(eta[b], g[b].G1, mu * g[b].G2));
            const double F2 = fma(eta[b], g[b].G0, fma(-beta[b], r0[b], mu) * g[b].G1);
            const double ir = rcp_f64<false>(r);
            const double d1 = F * ir;
            const double c = (0.5 * d1) * (F2 * ir);
            hc = max(hc, abs_hi(c));
            const double dX = fma(d1, c, d1);
            X[b] -= dX;
            d[b] = -dX;
            const int hx = abs_hi(X[b]);
            t1 = max(t1, abs_hi(dX) - hx);  // |dX| <= 2^-18 |X|  <=>  high words differ by at least 18 << 20
            hX = max(hX, hx);
        }
    }
    const bool redo = (hcorr >= 0x3fd00000) | (hz >= kHi0p1) | (hc >= kHi0p1) | (t1 > -0x01200000) | (hX >= kHiInf);

    if (__builtin_expect(__ballot_sync(amask, redo) != 0u, 0)) {  // warp-uniform, rarely taken
        if (redo) {
            KeplerLane<B> s;
#pragma unroll
            for (int b = 0; b < B; ++b) s.r0[b] = r0[b], s.ir0[b] = ir0[b], s.eta[b] = eta[b], s.beta[b] = beta[b];
            kepler_general_solve<B>(s, mu, tau);
#pragma unroll
            for (int b = 0; b < B; ++b) X[b] = s.X[b], d[b] = s.d[b], g[b] = s.g[b];
        }
    }
#pragma unroll
    for (int b = 0; b < B; ++b) {
        // G_n(X + d) to second order in d
        const double hd = 0.5 * d[b], bg1 = beta[b] * g[b].G1, bg0 = beta[b] * g[b].G0;
        const double G3 = fma(d[b], fma(hd, g[b].G1, g[b].G2), g[b].G3);
        const double G2 = fma(d[b], fma(hd, g[b].G0, g[b].G1), g[b].G2);
        const double G1 = fma(d[b], fma(-hd, bg1, g[b].G0), g[b].G1);
        const double G0 = fma(-d[b], fma(hd, bg0, bg1), g[b].G0);
        const double r = fma(r0[b], G0, fma(eta[b], G1, mu * G2));
        const double ir = rcp_f64<true>(r);
        const double mG2 = mu * G2;
        const double f = fma(-mG2, ir0[b], 1.0);
        const double gg = fma(-mu, G3, tau);
        const double fd = -(mu * G1) * (ir0[b] * ir);
        const double gd = fma(-mG2, ir, 1.0);
        if (valid(b)) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double qn = fma(f, Q[b][c], gg * P[b][c]);
                const double pn = fma(fd, Q[b][c], gd * P[b][c]);
                Q[b][c] = qn;
                P[b][c] = pn;
            }
        }
    }
}

// sum over the planets of the system of m_k W_k (W = V or Q).  L = 1: ascending k, the oracle's order.
// L > 1: per-lane partial sums, gathered from the lanes of the system in lane order.
template <int L, int B>
__device__ __forceinline__ void mass_weighted_sum(const double (&W)[B][3], const double (&m)[B], double (&out)[3], int l,
                                                  int base, unsigned amask) {
    double part[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int b = 0; b < B; ++b)
#pragma unroll
        for (int c = 0; c < 3; ++c) part[c] = fma(m[b], W[b][c], part[c]);  // dummy slots have m = 0
    if constexpr (L == 1) {
#pragma unroll
        for (int c = 0; c < 3; ++c) out[c] = part[c];
    } else {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double acc = __shfl_sync(amask, part[c], base);
#pragma unroll
            for (int i = 1; i < L; ++i) acc += __shfl_sync(amask, part[c], base + i);
            out[c] = acc;
        }
    }
}

// MAXREG caps the registers per thread (and with them the resident warps per SM) directly: __launch_bounds__'s
// minBlocks lets ptxas round down to a register count that spills.  Blocks must not exceed 65536 / MAXREG threads.
// MERGED = true (ENS_MVS_MERGED): the adjacent half sub-steps of consecutive steps are merged.  The
// closing half drift of step k and the opening one of step k+1 use the same drift velocity (one full drift), and the
// kick commutes with the Cartesian drift (the planets' mutual accelerations carry no net momentum, so the drift
// velocity is the same before and after a kick; the drift moves all planets alike, so A is unchanged): the two
// half kicks around the merged drift are one full kick.  A step is then  Kepler drift | A | full kick | full drift,
// opened by half drift + half kick and closed by half kick + half drift when the system leaves the loop.  The
// post-step positions Alg. 1 shows the monitors are formed as temporaries.  Same map in exact arithmetic; rounding
// differs from the unmerged kernel and oracle (tests/test_gpu_mvs_merged.py states the distance).
template <int N, int L, int B, int MAXREG, bool MERGED = false>
__global__ void __maxnreg__(MAXREG) mvs_kernel(View e, StepArgs p) {
    constexpr int P = N - 1;   // planets; body 0 is the star
    constexpr int S = 32 / L;  // systems per warp
    constexpr bool PADDED = (L * B != P);
    const int lane = threadIdx.x & 31;
    const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int sl = lane / L;
    const int l = lane - sl * L;
    const int base = sl * L;
    const int64_t sys = warp * S + sl;
    const bool live = (sl < S) && (sys < e.n_sys);
    extern __shared__ double2 ring_smem[];  // acc_ring_smem_words<L, B>() per warp (nothing for L = 1)
    double2* const W = ring_smem + (threadIdx.x >> 5) * acc_ring_smem_words<L, B>();

    double Q[B][3], V[B][3], A[B][3], m[B];
    double Xcm[3] = {0.0, 0.0, 0.0}, Vcm[3] = {0.0, 0.0, 0.0};
    // time folded with the direction of the run (ts = t forward, -t backward: exact), end test ts < p.te either way
    const bool fwd = p.dt > 0.0;
    double m0 = 1.0, im0 = 1.0, Mtot = 1.0, ts = 0.0;
    int st = ENS_STOP_NONFINITE;
    bool active = false;
#pragma unroll
    for (int b = 0; b < B; ++b) {
        // dummy slot (padded shapes only): massless, far from everything and from each other; never drifted
        Q[b][0] = 1.0e8 * (double)(l * B + b + 2);
        Q[b][1] = Q[b][2] = 0.0;
        V[b][0] = V[b][1] = V[b][2] = 0.0;
        m[b] = 0.0;
    }
    if (live) {
        st = e.status[sys];
        active = st < ENS_STOP_CLOSE;  // STOP_* are sticky; DONE_* run again
        ts = fwd ? e.time[sys] : -e.time[sys];
        // to_dh: total mass and centre of mass over all bodies in index order; every lane of the system reads all
        // bodies (L1-resident, once per launch) so that the sums need no communication
        double x0[3], sx[3] = {0.0, 0.0, 0.0}, sv[3] = {0.0, 0.0, 0.0};
        Mtot = 0.0;
#pragma unroll
        for (int i = 0; i < N; ++i) {
            const double mi = e.mass[(int64_t)i * e.n_pad + sys];
            Mtot += mi;
            if (i == 0) m0 = mi;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double xi = e.pos[(int64_t)(i * 3 + c) * e.n_pad + sys];
                const double vi = e.vel[(int64_t)(i * 3 + c) * e.n_pad + sys];
                if (i == 0) x0[c] = xi;
                sx[c] = fma(mi, xi, sx[c]);
                sv[c] = fma(mi, vi, sv[c]);
            }
        }
        im0 = 1.0 / m0;  // one IEEE divide per launch; the step loop multiplies (<= 1 ulp from the oracle's s / m0)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            Xcm[c] = sx[c] / Mtot;
            Vcm[c] = sv[c] / Mtot;
        }
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const int body = l * B + b + 1;
            if (!PADDED || body < N) {
                m[b] = e.mass[(int64_t)body * e.n_pad + sys];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    Q[b][c] = e.pos[(int64_t)(body * 3 + c) * e.n_pad + sys] - x0[c];
                    V[b][c] = e.vel[(int64_t)(body * 3 + c) * e.n_pad + sys] - Vcm[c];
                }
            }
        }
    }
    const bool writeback = active;

    const double h = p.dt, hh = p.hh;
    const bool mon_close = p.rc2_bits != 0ull;
    const bool mon_eject = p.re2_bits < 0x7FEFFFFFFFFFFFFFull;
    int64_t k = 0;
    unsigned r2min = ~0u;  // high word of the smallest planet-pair r^2 of the last acceleration evaluation
    double s[3] = {0.0, 0.0, 0.0};

    // Alg. 1 loop test before the first step (R10): time first, then the step budget
    if (active) {
        if (!(ts < p.te)) {
            st = ENS_DONE_TIME;
            active = false;
        } else if (k >= p.max_steps) {
            st = ENS_DONE_STEPS;
            active = false;
        }
    }
    {  // prepare(P) (Alg. 1): accelerations and drift velocity of the initial state
        const unsigned amask = __ballot_sync(0xffffffffu, active);
        if (active) {
            eval_acc_planets<P, L, B>(Q, m, A, r2min, l, base, amask, W);
            mass_weighted_sum<L, B>(V, m, s, l, base, amask);
#pragma unroll
            for (int c = 0; c < 3; ++c) s[c] = s[c] * im0;
        }
    }

    if constexpr (MERGED) {
        if (active) {  // open: half drift, half kick
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double sh = hh * s[c];
#pragma unroll
                for (int b = 0; b < B; ++b) {
                    Q[b][c] += sh;
                    V[b][c] = fma(hh, A[b][c], V[b][c]);
                }
                Xcm[c] = fma(hh, Vcm[c], Xcm[c]);
            }
        }
    }
    // The step loop.  All systems of the warp that run enter it together (mask `am`); a system leaves it through the
    // exact stop logic, which runs only when the quick test at the end of a step fails for some lane of the warp: the
    // loop itself carries one vote and one warp-uniform, almost never taken branch per step.
    const unsigned amask0 = __ballot_sync(0xffffffffu, active);
    if (active) {
        unsigned am = amask0;
        while (true) {
            // bookkeeping first: nothing below needs it before the tests at the end of the step
            ts += fabs(h);
            ++k;
            double Qp[B][3], Xp[3];  // MERGED: post-step positions (after the closing half drift), temporaries
            if constexpr (!MERGED) {
                // 1 + 2: Cartesian half drift, half kick
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const double sh = hh * s[c];
#pragma unroll
                    for (int b = 0; b < B; ++b) {
                        Q[b][c] += sh;
                        V[b][c] = fma(hh, A[b][c], V[b][c]);
                    }
                    Xcm[c] = fma(hh, Vcm[c], Xcm[c]);
                }
            }
            // 3: Kepler drift of every planet about mu = G m_0 (G = 1)
            kepler_drift_all<B>(Q, V, m0, h, am, [&](int b) { return !PADDED || (l * B + b < P); });
            if constexpr (MERGED) {
                // drift velocity of the rest of this step and the start of the next: kicks do not change it
                mass_weighted_sum<L, B>(V, m, s, l, base, am);
#pragma unroll
                for (int c = 0; c < 3; ++c) s[c] = s[c] * im0;
            }
            // 4: planet-planet accelerations at the new positions, half kick
            eval_acc_planets<P, L, B>(Q, m, A, r2min, l, base, am, W);
            if constexpr (!MERGED) {
#pragma unroll
                for (int b = 0; b < B; ++b)
#pragma unroll
                    for (int c = 0; c < 3; ++c) V[b][c] = fma(hh, A[b][c], V[b][c]);
                // 5: Cartesian half drift with the new momenta
                mass_weighted_sum<L, B>(V, m, s, l, base, am);
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    s[c] = s[c] * im0;
                    const double sh = hh * s[c];
#pragma unroll
                    for (int b = 0; b < B; ++b) Q[b][c] += sh;
                    Xcm[c] = fma(hh, Vcm[c], Xcm[c]);
                }
            } else {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const double sh = hh * s[c];
#pragma unroll
                    for (int b = 0; b < B; ++b) Qp[b][c] = Q[b][c] + sh;
                    Xp[c] = fma(hh, Vcm[c], Xcm[c]);
                }
            }
            const double(&Qm)[B][3] = MERGED ? Qp : Q;  // the post-step positions
            const double(&Xm)[3] = MERGED ? Xp : Xcm;

            // Monitors on the post-step state (Alg. 1 execute(M); R11) and the loop tests.  One quick test per
            // step on the integer ALU (high words): planet pairs farther apart than r_close (r2min of the acceleration
            // evaluation: the drift shifts every planet alike), every planet with some |Q_c| > r_close (farther
            // than that from the star), every |Q_c| < ce / 4 and |Xcm_c| < ce / 2 (then every barycentric coordinate is
            // below ce = r_eject / sqrt(3), and everything is finite), time left, steps left.  The exact logic runs only
            // when some lane of the warp fails it (warp-uniform, rarely taken).
            unsigned qhi = 0u, qlo = ~0u;
#pragma unroll
            for (int b = 0; b < B; ++b) {
                if (!PADDED || (l * B + b < P)) {
                    const unsigned m3 = max(max((unsigned)__double2hiint(Qm[b][0]) & 0x7fffffffu,
                                                (unsigned)__double2hiint(Qm[b][1]) & 0x7fffffffu),
                                            (unsigned)__double2hiint(Qm[b][2]) & 0x7fffffffu);
                    qhi = max(qhi, m3);
                    qlo = min(qlo, m3);
                }
            }
            const unsigned xhi = max(max((unsigned)__double2hiint(Xm[0]) & 0x7fffffffu, (unsigned)__double2hiint(Xm[1]) & 0x7fffffffu),
                                     (unsigned)__double2hiint(Xm[2]) & 0x7fffffffu);
            const bool go = (r2min > (unsigned)(p.rc2_bits >> 32)) && (qlo > p.rc1_hi) && (qhi < p.ceq_hi) &&
                            (xhi < p.cex_hi) && (ts < p.te) && (k < p.max_steps);
            if (__builtin_expect(__ballot_sync(am, !go) != 0u, 0)) {
                int f = 0;
                if (mon_close && pair_r2min<P, L, B>(Qm, l, base, am) < p.rc2_bits) f |= 1;
                u64 q2max = 0ull, q2min = ~0ull;  // over this lane's planets: star-planet separation is |Q_i|
#pragma unroll
                for (int b = 0; b < B; ++b) {
                    if (!PADDED || (l * B + b < P)) {
                        const u64 q2 = dbits(fma(Qm[b][2], Qm[b][2], fma(Qm[b][1], Qm[b][1], Qm[b][0] * Qm[b][0])));
                        q2max = q2 > q2max ? q2 : q2max;
                        q2min = q2 < q2min ? q2 : q2min;
                    }
                }
                if (q2max > 0x7FEFFFFFFFFFFFFFull) f |= 4;  // +inf or NaN
                if (q2min < p.rc2_bits) f |= 1;
                if (mon_eject) {  // distances from the coordinate origin need the star's barycentric position
                    double sq[3], x0[3];
                    mass_weighted_sum<L, B>(Qm, m, sq, l, base, am);
#pragma unroll
                    for (int c = 0; c < 3; ++c) x0[c] = Xm[c] - sq[c] / Mtot;
                    if (dbits(fma(x0[2], x0[2], fma(x0[1], x0[1], x0[0] * x0[0]))) > p.re2_bits) f |= 2;
#pragma unroll
                    for (int b = 0; b < B; ++b) {
                        if (!PADDED || (l * B + b < P)) {
                            const double xx = x0[0] + Qm[b][0], yy = x0[1] + Qm[b][1], zz = x0[2] + Qm[b][2];
                            if (dbits(fma(zz, zz, fma(yy, yy, xx * xx))) > p.re2_bits) f |= 2;
                        }
                    }
                }
                if constexpr (L > 1) {
                    int g = f;
#pragma unroll
                    for (int i = 1; i < L; ++i) {
                        int li = l + i;
                        if (li >= L) li -= L;
                        g |= __shfl_sync(am, f, base + li);
                    }
                    f = g;
                }
                if (f) {
                    st = (f & 4) ? ENS_STOP_NONFINITE : (f & 1) ? ENS_STOP_CLOSE : ENS_STOP_EJECT;
                    active = false;
                } else if (!(ts < p.te)) {
                    st = ENS_DONE_TIME;
                    active = false;
                } else if (k >= p.max_steps) {
                    st = ENS_DONE_STEPS;
                    active = false;
                }
                am = __ballot_sync(am, active);  // the systems that go on
                if (!active) {
                    if constexpr (MERGED) {  // the system leaves the loop: close the step
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
#pragma unroll
                            for (int b = 0; b < B; ++b) {
                                V[b][c] = fma(hh, A[b][c], V[b][c]);
                                Q[b][c] = Qp[b][c];
                            }
                            Xcm[c] = Xp[c];
                        }
                    }
                    break;
                }
            }
            if constexpr (MERGED) {  // full kick and full drift: the closing halves of this step and the opening ones of the next
#pragma unroll
                for (int c = 0; c < 3; ++c) {
#pragma unroll
                    for (int b = 0; b < B; ++b) {
                        V[b][c] = fma(h, A[b][c], V[b][c]);
                        Q[b][c] = fma(h, s[c], Q[b][c]);
                    }
                    Xcm[c] = fma(h, Vcm[c], Xcm[c]);
                }
            }
        }
    }

    // from_dh and store.  All lanes of a system left the loop together (t, k and the monitor flags are replicated).
    const unsigned wmask = __ballot_sync(0xffffffffu, writeback);
    if (writeback) {
        double sq[3], sp[3], x0[3], v0[3];
        mass_weighted_sum<L, B>(Q, m, sq, l, base, wmask);
        mass_weighted_sum<L, B>(V, m, sp, l, base, wmask);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            x0[c] = Xcm[c] - sq[c] / Mtot;
            v0[c] = Vcm[c] - sp[c] / m0;
        }
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const int body = l * B + b + 1;
            if (!PADDED || body < N) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    e.pos[(int64_t)(body * 3 + c) * e.n_pad + sys] = x0[c] + Q[b][c];
                    e.vel[(int64_t)(body * 3 + c) * e.n_pad + sys] = V[b][c] + Vcm[c];
                }
            }
        }
        if (l == 0) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                e.pos[(int64_t)c * e.n_pad + sys] = x0[c];
                e.vel[(int64_t)c * e.n_pad + sys] = v0[c];
            }
            e.time[sys] = fwd ? ts : -ts;
            e.status[sys] = st;
            e.nsteps[sys] += k;
        }
    }
}

}  // namespace ensd
