// ens_oracle.cpp — CPU ORACLE for the ensemble Hermite / MVS step loop of Swarm-NG (arxiv 1208.1157).
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may build, load or call anything under oracle/.  It shares no code
// (headers, helpers, tables, constants) with paper_1208_1157_b200/csrc and neither side includes the other.
//
// Plain, slow, one system at a time, IEEE double (prec=0) or x87 80-bit long double (prec=1, the noise
// reference), correctly rounded sqrt and divide, no fast-math, compiled with -ffp-contract=off.
// It follows PAPER.md (`P:L<n>` = /root/reference/PAPER.md line n) step by step, with the readings
// R1..R15, R-M1..R-M7 of DESIGN.md §3 where the extracted text is garbled or silent.
//
// Layout of every array argument: C order, pos/vel [n_sys][n_body][3], mass [n_sys][n_body], per-system
// arrays [n_sys].  Body 0 is the central body.  G = 1.
//
// Pins (tests/test_oracle_*.py, tests/test_golden.py): 2-body closed forms, Kepler's equation, order-4 / order-2
// convergence, symmetric-corrector identity, reversal, invariants, finite-difference jerk, brute-force sums, Stumpff
// closed forms, test-particle exactness of the Kepler drift, hand-built monitor crossings; adaptive step (Eq. 5):
// circular and apsidal closed forms dt = tau / (w sqrt 2), scaling laws, order 4 in tau; 2-evaluation Hermite: order
// 4, first step identical to the 3-evaluation step; Cash-Karp: all 17 rooted-tree order conditions on the tableau,
// measured order 5 (embedded: 4); the Kepler solver's bracket-and-bisect fallback: cases that reach it against Kepler's
// equation (elliptic, multi-revolution) and against orbit invariants, the hyperbolic Kepler equation and the group
// property (hyperbolic); adaptive Cash-Karp: convergence to Kepler's equation at the rate the control implies, the
// control's definition on single trial steps, rejected steps leaving the state untouched; merged MVS: one step
// bit-identical to the unmerged step, same order-2 convergence and invariants.  The whole file runs clean under
// AddressSanitizer + UBSan (tests/test_oracle_sanitize.py).  No function in this file is "parity unpinned"; the only
// unpinned item is the paper's Table 1, whose orbital phases are unspecified.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

namespace {

enum { ST_ACTIVE = 0, ST_DONE_TIME = 1, ST_DONE_STEPS = 2, ST_STOP_CLOSE = 3, ST_STOP_EJECT = 4, ST_STOP_NONFINITE = 5, ST_STOP_STEPSIZE = 6 };

template <class R> inline R rsqrt_exact(R r2) { return R(1) / std::sqrt(r2); }

// ---------------------------------------------------------------------------------------------------
// Acceleration and jerk.  Eq. 1 (denominator read as |x_j - x_i|^3, R1) and its time derivative
// ("analytic expressions", R2):   a_i = sum_k m_k dx / r^3,   j_i = sum_k m_k [dv/r^3 - 3 (dx.dv) dx / r^5].
// Summation order: planets k = 1..n-1 ascending, the star (body 0) LAST (R7).
// ---------------------------------------------------------------------------------------------------
template <class R>
void eval_acc_jerk(int n, const R* x, const R* v, const R* m, R* a, R* j) {
    for (int i = 0; i < n; ++i) {
        R ai[3] = {0, 0, 0}, ji[3] = {0, 0, 0};
        for (int kk = 1; kk <= n; ++kk) {
            const int k = (kk == n) ? 0 : kk;  // 1, 2, ..., n-1, then 0
            if (k == i) continue;
            R dx[3], dv[3];
            for (int c = 0; c < 3; ++c) {
                dx[c] = x[3 * k + c] - x[3 * i + c];
                dv[c] = v[3 * k + c] - v[3 * i + c];
            }
            const R r2 = dx[0] * dx[0] + dx[1] * dx[1] + dx[2] * dx[2];
            const R rv = dx[0] * dv[0] + dx[1] * dv[1] + dx[2] * dv[2];
            const R rinv = rsqrt_exact(r2);
            const R rinv3 = rinv * rinv * rinv;
            for (int c = 0; c < 3; ++c) {
                ai[c] += m[k] * rinv3 * dx[c];
                ji[c] += m[k] * rinv3 * (dv[c] - R(3) * (rv / r2) * dx[c]);
            }
        }
        for (int c = 0; c < 3; ++c) {
            a[3 * i + c] = ai[c];
            j[3 * i + c] = ji[c];
        }
    }
}

// Acceleration only, planets on planets, in heliocentric positions Q (index 1..n-1); the star-planet
// term is excluded because the Kepler drift carries it.
template <class R>
void eval_acc_planets(int n, const R* Q, const R* m, R* A) {
    for (int i = 1; i < n; ++i) {
        R ai[3] = {0, 0, 0};
        for (int k = 1; k < n; ++k) {
            if (k == i) continue;
            R dx[3];
            for (int c = 0; c < 3; ++c) dx[c] = Q[3 * k + c] - Q[3 * i + c];
            const R r2 = dx[0] * dx[0] + dx[1] * dx[1] + dx[2] * dx[2];
            const R rinv = rsqrt_exact(r2);
            const R rinv3 = rinv * rinv * rinv;
            for (int c = 0; c < 3; ++c) ai[c] += m[k] * rinv3 * dx[c];
        }
        for (int c = 0; c < 3; ++c) A[3 * i + c] = ai[c];
    }
}

// ---------------------------------------------------------------------------------------------------
// One Hermite step, Alg. 2 with Eq. 3 and Eq. 4 read as R3-R6:
//   three evaluations per step: (a0,j0) at the current state, then two corrector iterations
//   (P:L89), each re-evaluating (a_k,j_k) at the latest iterate; corrector base is the PREDICTED x_p,v_p,
//   coefficient of (a0-a_k) h^2 is 3/20.
// ---------------------------------------------------------------------------------------------------
template <class R>
void hermite_step(int n, R* x, R* v, const R* m, R h, int n_corr = 2) {
    const int d = 3 * n;
    std::vector<R> a0(d), j0(d), a1(d), j1(d), xp(d), vp(d), xc(d), vc(d);
    eval_acc_jerk(n, x, v, m, a0.data(), j0.data());
    for (int q = 0; q < d; ++q) {
        xp[q] = x[q] + v[q] * h + a0[q] * (h * h) / R(2) + j0[q] * (h * h * h) / R(6);
        vp[q] = v[q] + a0[q] * h + j0[q] * (h * h) / R(2);
        xc[q] = xp[q];
        vc[q] = vp[q];
    }
    for (int it = 0; it < n_corr; ++it) {
        eval_acc_jerk(n, xc.data(), vc.data(), m, a1.data(), j1.data());
        for (int q = 0; q < d; ++q) {
            xc[q] = xp[q] - (R(3) / R(20)) * (a0[q] - a1[q]) * (h * h) - (R(1) / R(60)) * (R(7) * j0[q] + R(2) * j1[q]) * (h * h * h);
            vc[q] = vp[q] - (R(1) / R(2)) * (a0[q] - a1[q]) * h - (R(1) / R(12)) * (R(5) * j0[q] + j1[q]) * (h * h);
        }
    }
    for (int q = 0; q < d; ++q) {
        x[q] = xc[q];
        v[q] = vc[q];
    }
}

// ---------------------------------------------------------------------------------------------------
// Alg. 2 exactly as printed: TWO evaluations per step.  a^(0), j^(0) are inputs of the step, and the
// loop leaves a^(2), j^(2) (evaluated at the iterate x^(2), v^(2), i.e. before the last correction) behind; the
// next step takes them as its a^(0), j^(0) (reading R6-alt: "carry").  Coefficients and bases as in hermite_step
// (R3-R5).  a0, j0: in = values for this step, out = values for the next one.
// ---------------------------------------------------------------------------------------------------
template <class R>
void hermite_step_carry(int n, R* x, R* v, const R* m, R h, R* a0, R* j0) {
    const int d = 3 * n;
    std::vector<R> a1(d), j1(d), xp(d), vp(d), xc(d), vc(d);
    for (int q = 0; q < d; ++q) {
        xp[q] = x[q] + v[q] * h + a0[q] * (h * h) / R(2) + j0[q] * (h * h * h) / R(6);
        vp[q] = v[q] + a0[q] * h + j0[q] * (h * h) / R(2);
        xc[q] = xp[q];
        vc[q] = vp[q];
    }
    for (int it = 0; it < 2; ++it) {
        eval_acc_jerk(n, xc.data(), vc.data(), m, a1.data(), j1.data());
        for (int q = 0; q < d; ++q) {
            xc[q] = xp[q] - (R(3) / R(20)) * (a0[q] - a1[q]) * (h * h) - (R(1) / R(60)) * (R(7) * j0[q] + R(2) * j1[q]) * (h * h * h);
            vc[q] = vp[q] - (R(1) / R(2)) * (a0[q] - a1[q]) * h - (R(1) / R(12)) * (R(5) * j0[q] + j1[q]) * (h * h);
        }
    }
    for (int q = 0; q < d; ++q) {
        x[q] = xc[q];
        v[q] = vc[q];
        a0[q] = a1[q];
        j0[q] = j1[q];
    }
}

// ---------------------------------------------------------------------------------------------------
// Fixed-step Runge-Kutta Cash-Karp (section 2.2.2, section 4.3.2): the explicit six-stage
// embedded 4(5) pair of Cash & Karp (1990) applied to y = (x, v), y' = (v, a(x)); accelerations only, "six sub-steps
// and six force evaluations for each step".  The step propagates the FIFTH-order solution, as the GSL rkck
// stepper the paper says it follows does (reading R-RK1); the embedded fourth-order solution only serves the error
// estimate err = y5 - y4 (returned for the tests; the adaptive controller is not defined by the paper: out of
// scope).
// ---------------------------------------------------------------------------------------------------
template <class R>
struct CashKarp {
    R c[6], a[6][5], b5[6], b4[6];
    CashKarp() {
        const R z = 0;
        const R cc[6] = {z, R(1) / 5, R(3) / 10, R(3) / 5, R(1), R(7) / 8};
        const R aa[6][5] = {{z, z, z, z, z},
                            {R(1) / 5, z, z, z, z},
                            {R(3) / 40, R(9) / 40, z, z, z},
                            {R(3) / 10, R(-9) / 10, R(6) / 5, z, z},
                            {R(-11) / 54, R(5) / 2, R(-70) / 27, R(35) / 27, z},
                            {R(1631) / 55296, R(175) / 512, R(575) / 13824, R(44275) / 110592, R(253) / 4096}};
        const R bb5[6] = {R(37) / 378, z, R(250) / 621, R(125) / 594, z, R(512) / 1771};
        const R bb4[6] = {R(2825) / 27648, z, R(18575) / 48384, R(13525) / 55296, R(277) / 14336, R(1) / 4};
        for (int i = 0; i < 6; ++i) {
            c[i] = cc[i];
            b5[i] = bb5[i];
            b4[i] = bb4[i];
            for (int k = 0; k < 5; ++k) a[i][k] = aa[i][k];
        }
    }
};

template <class R>
void eval_acc(int n, const R* x, const R* m, R* a) {  // Eq. 1 (R1), planets ascending then the star
    for (int i = 0; i < n; ++i) {
        R ai[3] = {0, 0, 0};
        for (int kk = 1; kk <= n; ++kk) {
            const int k = (kk == n) ? 0 : kk;
            if (k == i) continue;
            R dx[3];
            for (int c = 0; c < 3; ++c) dx[c] = x[3 * k + c] - x[3 * i + c];
            const R r2 = dx[0] * dx[0] + dx[1] * dx[1] + dx[2] * dx[2];
            const R rinv = rsqrt_exact(r2);
            const R rinv3 = rinv * rinv * rinv;
            for (int c = 0; c < 3; ++c) ai[c] += m[k] * rinv3 * dx[c];
        }
        for (int c = 0; c < 3; ++c) a[3 * i + c] = ai[c];
    }
}

// one step; errx / errv (may be null) receive y5 - y4
template <class R>
void rkck_step(int n, R* x, R* v, const R* m, R h, R* errx = nullptr, R* errv = nullptr) {
    static const CashKarp<R> T;
    const int d = 3 * n;
    std::vector<R> kx(6 * d), kv(6 * d), xs(d), vs(d);
    for (int i = 0; i < 6; ++i) {
        for (int q = 0; q < d; ++q) {
            R sx = 0, sv = 0;
            for (int k = 0; k < i; ++k) {
                sx += T.a[i][k] * kx[k * d + q];
                sv += T.a[i][k] * kv[k * d + q];
            }
            xs[q] = x[q] + h * sx;
            vs[q] = v[q] + h * sv;
        }
        for (int q = 0; q < d; ++q) kx[i * d + q] = vs[q];      // x' = v
        eval_acc(n, xs.data(), m, kv.data() + i * d);           // v' = a(x)
    }
    for (int q = 0; q < d; ++q) {
        R x5 = 0, v5 = 0, x4 = 0, v4 = 0;
        for (int i = 0; i < 6; ++i) {
            x5 += T.b5[i] * kx[i * d + q];
            v5 += T.b5[i] * kv[i * d + q];
            x4 += T.b4[i] * kx[i * d + q];
            v4 += T.b4[i] * kv[i * d + q];
        }
        if (errx) errx[q] = h * (x5 - x4);
        if (errv) errv[q] = h * (v5 - v4);
        x[q] += h * x5;
        v[q] += h * v5;
    }
}

// ---------------------------------------------------------------------------------------------------
// Adaptive time step, Eq. 5:  dt = tau [ sum_i |j_i0|^2 / |a_i0|^2 ]^(-1/2),  i over ALL bodies of the
// system ("i indexes a body in the system", the star included: reading R-A1), a_i0 and j_i0 evaluated at the
// beginning of the step ("uses only the values at the beginning of the time step").  tau carries the
// sign of the integration direction.  A body with |a|^2 = 0 (no other mass in the system) contributes nothing
// (reading R-A2).  The step itself is hermite_step with this dt (same three evaluations, R6).
// ---------------------------------------------------------------------------------------------------
template <class R>
R hermite_adaptive_dt(int n, const R* x, const R* v, const R* m, R tau) {
    std::vector<R> a(3 * n), j(3 * n);
    eval_acc_jerk(n, x, v, m, a.data(), j.data());
    R sum = 0;
    for (int i = 0; i < n; ++i) {
        const R a2 = a[3 * i] * a[3 * i] + a[3 * i + 1] * a[3 * i + 1] + a[3 * i + 2] * a[3 * i + 2];
        const R j2 = j[3 * i] * j[3 * i] + j[3 * i + 1] * j[3 * i + 1] + j[3 * i + 2] * j[3 * i + 2];
        if (a2 > R(0)) sum += j2 / a2;
    }
    return tau / std::sqrt(sum);
}

// ---------------------------------------------------------------------------------------------------
// Monitors (Alg. 1 `execute(M)` after `advance(P)`; thresholds from BASELINE.json;
// reading R11).  Evaluated on the post-step state only.  Order: non-finite, close approach, ejection.
// ---------------------------------------------------------------------------------------------------
template <class R>
int monitors(int n, const R* x, double r_close, double r_eject) {
    for (int i = 0; i < n; ++i) {
        const R d2 = x[3 * i] * x[3 * i] + x[3 * i + 1] * x[3 * i + 1] + x[3 * i + 2] * x[3 * i + 2];
        if (!std::isfinite((double)d2)) return ST_STOP_NONFINITE;
    }
    if (r_close > 0) {
        for (int i = 0; i < n; ++i)
            for (int k = i + 1; k < n; ++k) {
                R dx[3];
                for (int c = 0; c < 3; ++c) dx[c] = x[3 * k + c] - x[3 * i + c];
                const R r = std::sqrt(dx[0] * dx[0] + dx[1] * dx[1] + dx[2] * dx[2]);
                if (r < R(r_close)) return ST_STOP_CLOSE;
            }
    }
    if (std::isfinite(r_eject) && r_eject > 0) {
        for (int i = 0; i < n; ++i) {
            const R d = std::sqrt(x[3 * i] * x[3 * i] + x[3 * i + 1] * x[3 * i + 1] + x[3 * i + 2] * x[3 * i + 2]);
            if (d > R(r_eject)) return ST_STOP_EJECT;
        }
    }
    return ST_ACTIVE;
}

inline bool time_left(double dt, double t, double t_end) {
    // direction-aware `t < t_end` (R10): continue while sign(dt) * (t_end - t) > 0; no clipping of the last step.
    return dt > 0 ? (t < t_end) : (t > t_end);
}

// ---------------------------------------------------------------------------------------------------
// Energy and angular momentum.  Eq. 6 with each unordered pair counted once (R9).
// ---------------------------------------------------------------------------------------------------
template <class R>
void energy_L(int n, const R* x, const R* v, const R* m, R* E, R* L) {
    R ke = 0, pe = 0;
    for (int i = 0; i < n; ++i) ke += R(0.5) * m[i] * (v[3 * i] * v[3 * i] + v[3 * i + 1] * v[3 * i + 1] + v[3 * i + 2] * v[3 * i + 2]);
    for (int i = 0; i < n; ++i)
        for (int k = i + 1; k < n; ++k) {
            R dx[3];
            for (int c = 0; c < 3; ++c) dx[c] = x[3 * k + c] - x[3 * i + c];
            pe -= m[i] * m[k] / std::sqrt(dx[0] * dx[0] + dx[1] * dx[1] + dx[2] * dx[2]);
        }
    *E = ke + pe;
    if (L) {
        L[0] = L[1] = L[2] = 0;
        for (int i = 0; i < n; ++i) {
            const R* xi = x + 3 * i;
            const R* vi = v + 3 * i;
            L[0] += m[i] * (xi[1] * vi[2] - xi[2] * vi[1]);
            L[1] += m[i] * (xi[2] * vi[0] - xi[0] * vi[2]);
            L[2] += m[i] * (xi[0] * vi[1] - xi[1] * vi[0]);
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// Stumpff functions c0..c3 (c_n(z) = sum_k (-z)^k / (2k+n)!): series for |z| small, argument quartering
// otherwise (R-M3).  c0 = cos sqrt z, c1 = sin sqrt z / sqrt z, c2 = (1-c0)/z, c3 = (1-c1)/z for z > 0.
// ---------------------------------------------------------------------------------------------------
template <class R>
void stumpff(R z, R c[4]) {
    int nq = 0;
    while (std::fabs(z) > R(0.1)) {
        z /= R(4);
        ++nq;
    }
    // series c_n(z) = sum_k (-z)^k / (2k+n)!, 12 terms: |z|^12 / 26! is far below 1e-30 for |z| <= 0.1
    R t2 = R(1) / R(2), t3 = R(1) / R(6);  // k = 0 terms: 1/2!, 1/3!
    R c2 = t2, c3 = t3;
    for (int k = 1; k < 12; ++k) {
        t2 *= -z / R((2 * k + 1) * (2 * k + 2));
        t3 *= -z / R((2 * k + 2) * (2 * k + 3));
        c2 += t2;
        c3 += t3;
    }
    R c1 = R(1) - z * c3;
    R c0 = R(1) - z * c2;
    for (; nq > 0; --nq) {
        // c_n(4z) from c_n(z)
        const R n3 = (c2 + c0 * c3) / R(4);
        const R n2 = c1 * c1 / R(2);
        const R n1 = c0 * c1;
        const R n0 = R(2) * c0 * c0 - R(1);
        c3 = n3; c2 = n2; c1 = n1; c0 = n0;
    }
    c[0] = c0; c[1] = c1; c[2] = c2; c[3] = c3;
}

// ---------------------------------------------------------------------------------------------------
// Kepler drift of one body about a fixed centre of gravitational parameter mu for time tau,
// by universal variables (BASELINE.json config 4; R-M3, R-M4):
//   r0 = |q|, eta = q.p, beta = 2 mu / r0 - |p|^2;   solve  r0 G1 + eta G2 + mu G3 = tau  for X,
//   G_n = X^n c_n(beta X^2); Newton with derivative r = r0 G0 + eta G1 + mu G2; guess X = tau / r0.
//   f = 1 - mu G2 / r0, g = tau - mu G3, f' = -mu G1 / (r0 r), g' = 1 - mu G2 / r.
// Returns the number of Newton iterations (negative if the bisection fallback was needed).
// ---------------------------------------------------------------------------------------------------
template <class R>
struct GFun { R G0, G1, G2, G3; };

template <class R>
GFun<R> gfuncs(R beta, R X) {
    R c[4];
    stumpff(beta * X * X, c);
    GFun<R> G;
    G.G0 = c[0];
    G.G1 = X * c[1];
    G.G2 = X * X * c[2];
    G.G3 = X * X * X * c[3];
    return G;
}

template <class R>
int kepler_drift(R* q, R* p, R mu, R tau) {
    const R r0 = std::sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2]);
    const R eta = q[0] * p[0] + q[1] * p[1] + q[2] * p[2];
    const R v2 = p[0] * p[0] + p[1] * p[1] + p[2] * p[2];
    const R beta = R(2) * mu / r0 - v2;
    const R eps = std::is_same<R, double>::value ? R(1e-15) : R(1e-18);

    auto resid = [&](R X, GFun<R>& G) {
        G = gfuncs(beta, X);
        return r0 * G.G1 + eta * G.G2 + mu * G.G3 - tau;
    };

    R X = tau / r0;
    GFun<R> G;
    int iters = 0;
    bool ok = false;
    for (; iters < 50; ++iters) {
        const R F = resid(X, G);
        const R dF = r0 * G.G0 + eta * G.G1 + mu * G.G2;
        const R dX = F / dF;
        X -= dX;
        if (!(std::fabs(dX) > eps * std::fabs(X))) { ok = true; ++iters; break; }
    }
    if (!ok || !std::isfinite((double)X)) {
        // guaranteed-convergent fallback: the residual is monotone in X (dF/dX = r > 0); bracket and bisect.
        R lo = 0, hi = tau / r0;
        GFun<R> Gt;
        const R sgn = tau >= 0 ? R(1) : R(-1);
        if (hi == 0) hi = sgn;
        for (int k = 0; k < 200 && sgn * resid(hi, Gt) < 0; ++k) hi *= R(2);
        for (int k = 0; k < 200; ++k) {
            const R mid = R(0.5) * (lo + hi);
            if (sgn * resid(mid, Gt) < 0) lo = mid; else hi = mid;
        }
        X = R(0.5) * (lo + hi);
        iters = -iters;
    }
    G = gfuncs(beta, X);
    const R r = r0 * G.G0 + eta * G.G1 + mu * G.G2;
    const R f = R(1) - mu * G.G2 / r0;
    const R g = tau - mu * G.G3;
    const R fd = -mu * G.G1 / (r0 * r);
    const R gd = R(1) - mu * G.G2 / r;
    for (int c = 0; c < 3; ++c) {
        const R qn = f * q[c] + g * p[c];
        const R pn = fd * q[c] + gd * p[c];
        q[c] = qn;
        p[c] = pn;
    }
    return iters;
}

// ---------------------------------------------------------------------------------------------------
// MVS in democratic-heliocentric variables (R-M1): heliocentric positions Q_i = x_i - x_0, barycentric
// velocities V_i = v_i - V_cm (i >= 1), plus the centre of mass X_cm, V_cm.  Five sub-steps, unmerged
// (R-M7); mu = G m_0 (R-M2); planet-planet accelerations reused across the step boundary.
// ---------------------------------------------------------------------------------------------------
template <class R>
struct DH {
    int n;
    std::vector<R> Q, V, A;  // index 3*i+c, i = 1..n-1 (slot 0 unused)
    R Xcm[3], Vcm[3], M;
};

template <class R>
void to_dh(int n, const R* x, const R* v, const R* m, DH<R>& s) {
    s.n = n;
    s.Q.assign(3 * n, 0); s.V.assign(3 * n, 0); s.A.assign(3 * n, 0);
    s.M = 0;
    for (int i = 0; i < n; ++i) s.M += m[i];
    for (int c = 0; c < 3; ++c) {
        R sx = 0, sv = 0;
        for (int i = 0; i < n; ++i) { sx += m[i] * x[3 * i + c]; sv += m[i] * v[3 * i + c]; }
        s.Xcm[c] = sx / s.M;
        s.Vcm[c] = sv / s.M;
    }
    for (int i = 1; i < n; ++i)
        for (int c = 0; c < 3; ++c) {
            s.Q[3 * i + c] = x[3 * i + c] - x[c];
            s.V[3 * i + c] = v[3 * i + c] - s.Vcm[c];
        }
}

template <class R>
void from_dh(const DH<R>& s, const R* m, R* x, R* v) {
    const int n = s.n;
    for (int c = 0; c < 3; ++c) {
        R sq = 0, sp = 0;
        for (int k = 1; k < n; ++k) { sq += m[k] * s.Q[3 * k + c]; sp += m[k] * s.V[3 * k + c]; }
        x[c] = s.Xcm[c] - sq / s.M;
        if (v) v[c] = s.Vcm[c] - sp / m[0];
        for (int i = 1; i < n; ++i) {
            x[3 * i + c] = x[c] + s.Q[3 * i + c];
            if (v) v[3 * i + c] = s.V[3 * i + c] + s.Vcm[c];
        }
    }
}

template <class R>
void mvs_linear_drift(DH<R>& s, const R* m, R hh) {  // Cartesian drift
    for (int c = 0; c < 3; ++c) {
        R sp = 0;
        for (int k = 1; k < s.n; ++k) sp += m[k] * s.V[3 * k + c];
        const R sh = sp / m[0];
        for (int i = 1; i < s.n; ++i) s.Q[3 * i + c] += hh * sh;
        s.Xcm[c] += hh * s.Vcm[c];
    }
}

template <class R>
void mvs_kick(DH<R>& s, R hh) {
    for (int q = 3; q < 3 * s.n; ++q) s.V[q] += hh * s.A[q];
}

template <class R>
void mvs_step(DH<R>& s, const R* m, R h) {
    const R hh = h / R(2);
    mvs_linear_drift(s, m, hh);
    mvs_kick(s, hh);
    for (int i = 1; i < s.n; ++i) kepler_drift(&s.Q[3 * i], &s.V[3 * i], m[0], h);
    eval_acc_planets(s.n, s.Q.data(), m, s.A.data());
    mvs_kick(s, hh);
    mvs_linear_drift(s, m, hh);
}

// ---------------------------------------------------------------------------------------------------
// Adaptive-step Runge-Kutta Cash-Karp ("closely based on the gsl_odeiv2_step_rkck stepper ... one with an
// adaptive time-step"; "uses the Cash-Karp method at the end of the step to compute the 5th order error.  If
// the error exceeds the user specified accuracy parameter (eps), the step is rejected, e.g. positions, velocities and
// time are not updated ...  Instead, the next attempted time-step will use a smaller time-step").  The paper gives
// neither the error norm nor the step-size rule; reading R-RK2' takes the standard step-size
// control the GSL manual documents for that stepper family:
//   error level of a trial step   r = max( max|errx| / (eps X),  max|errv| / (eps V) ),   err = y5 - y4 of rkck_step,
//                                 X = max_b |x_b|_2, V = max_b |v_b|_2 of the state the step starts from (the scale of
//                                 reading R13; a per-component relative scale is undefined for the exact zeros of
//                                 coplanar initial conditions);
//   r > 1.1   reject: state and time untouched, h <- h max(1/5, F(S r^(-1/q))), try again;
//   else      accept (the fifth-order solution, R-RK1; t += h), and if r < 0.5 the NEXT step starts from
//             h <- h min(5, max(1, F(S r^(-1/(q+1)))));
//   S = 0.9, q = 4 (the manual's "consistency order, e.g. q = 4 for 4(5) embedded RK");
//   F(f) = floor(16 f) / 16: the factor is taken from a discrete set (the device the paper proposes for reproducible
//   adaptive steps, "choose from a discrete set of time steps").  The error estimate is a difference of nearly
//   equal sums, so r carries relative rounding noise of 1e-9..1e-7; with a continuous factor that noise would reach
//   every later step size and time, and two correct implementations would differ at the 1e-8 level after a few
//   hundred steps; with the discrete factor they take bit-identical steps unless r falls within the noise of a
//   boundary (rare, and then both step sequences are valid).
// h is the per-system trial step; every call starts it at the caller's dt (sign = direction).  No clipping of the
// last step (R10).  *accepted: 1 if the step was taken.  Returns the error level r.
// ---------------------------------------------------------------------------------------------------
template <class R>
R rkck_adaptive_trial(int n, R* x, R* v, const R* m, R& h, R eps, bool* accepted) {
    const int d = 3 * n;
    std::vector<R> xn(x, x + d), vn(v, v + d), ex(d), ev(d);
    rkck_step(n, xn.data(), vn.data(), m, h, ex.data(), ev.data());
    R X = 0, V = 0, EX = 0, EV = 0;
    for (int i = 0; i < n; ++i) {
        const R xx = std::sqrt(x[3 * i] * x[3 * i] + x[3 * i + 1] * x[3 * i + 1] + x[3 * i + 2] * x[3 * i + 2]);
        const R vv = std::sqrt(v[3 * i] * v[3 * i] + v[3 * i + 1] * v[3 * i + 1] + v[3 * i + 2] * v[3 * i + 2]);
        if (xx > X) X = xx;
        if (vv > V) V = vv;
    }
    for (int q = 0; q < d; ++q) {
        if (std::fabs(ex[q]) > EX) EX = std::fabs(ex[q]);
        if (std::fabs(ev[q]) > EV) EV = std::fabs(ev[q]);
    }
    const R rx = EX / (eps * X), rv = EV / (eps * V);
    const R r = rx > rv ? rx : rv;
    const R S = R(9) / R(10);
    if (r > R(11) / R(10)) {  // reject: nothing but h changes
        R f = std::floor(R(16) * (S * std::pow(r, R(-1) / R(4)))) / R(16);
        if (f < R(1) / R(5)) f = R(1) / R(5);
        h *= f;
        *accepted = false;
        return r;
    }
    for (int q = 0; q < d; ++q) { x[q] = xn[q]; v[q] = vn[q]; }
    *accepted = true;
    if (r < R(1) / R(2)) {
        R f = std::floor(R(16) * (S * std::pow(r, R(-1) / R(5)))) / R(16);
        if (f > R(5)) f = R(5);
        if (f < R(1)) f = R(1);
        h *= f;  // r = 0 gives f = inf -> 5
    }
    return r;
}

// ---------------------------------------------------------------------------------------------------
// The generic integrator loop, Alg. 1 with R10-R12:
//   while ACTIVE and steps_this_call < max_steps and time left: advance; ++nsteps; t += h; monitors;
//   exit status: STOP_* (sticky) | DONE_TIME (t reached t_end) | DONE_STEPS.
// ---------------------------------------------------------------------------------------------------
template <class R>
void run_system(int integrator, int n, double* pos, double* vel, const double* mass, double* time, int32_t* status,
                int64_t* nsteps, double dt, double t_end, int64_t max_steps, double r_close, double r_eject, int n_corr,
                double rk_eps = 1e-9, int64_t* nreject = nullptr) {
    if (*status >= ST_STOP_CLOSE) return;  // sticky until the state is set again
    std::vector<R> x(3 * n), v(3 * n), m(n);
    for (int q = 0; q < 3 * n; ++q) { x[q] = pos[q]; v[q] = vel[q]; }
    for (int i = 0; i < n; ++i) m[i] = mass[i];
    R t = *time;
    const R h = dt;
    int st = ST_ACTIVE;
    int64_t k = 0;
    DH<R> s;
    std::vector<R> xm(3 * n), ca(3 * n), cj(3 * n);
    if (integrator == 3)  // carried (a, j): evaluated once at the state the call starts from
        eval_acc_jerk(n, x.data(), v.data(), m.data(), ca.data(), cj.data());
    if (integrator == 1 || integrator == 5) {
        to_dh(n, x.data(), v.data(), m.data(), s);
        eval_acc_planets(n, s.Q.data(), m.data(), s.A.data());  // prepare(P)
    }
    if (integrator == 5) {
        // MVS with the adjacent half sub-steps of consecutive steps merged (P:L105-109 lists five sub-steps; P:L256:
        // "the separation between planets does not change during Cartesian drift and kick sub-steps").  The closing
        // half drift of step k and the opening one of step k+1 use the same drift velocity and are one full drift; the
        // kick commutes with the Cartesian drift (the planets' accelerations sum to zero momentum, so the drift velocity
        // is the same before and after a kick, and the drift moves every planet alike, so A is unchanged): the two half
        // kicks that surround the merged drift are one full kick.  In exact arithmetic every post-step state equals the
        // unmerged map's; rounding differs (the "parity cost", measured in tests/test_oracle_mvs_merged.py).
        //   open:  D(h/2) K(h/2)
        //   step:  Kepler(h); A = acc;  post-step state = K(h/2) D(h/2) of the current one (formed for the monitors
        //          and as the result when the loop ends here);  if the loop goes on: K(h) D(h) instead.
        const R hh = h / R(2);
        bool opened = false;
        DH<R> post;
        while (true) {
            if (!time_left(dt, (double)t, t_end)) { st = ST_DONE_TIME; break; }
            if (k >= max_steps) { st = ST_DONE_STEPS; break; }
            if (!opened) {
                mvs_linear_drift(s, m.data(), hh);
                mvs_kick(s, hh);
                opened = true;
            }
            for (int i = 1; i < n; ++i) kepler_drift(&s.Q[3 * i], &s.V[3 * i], m[0], h);
            eval_acc_planets(n, s.Q.data(), m.data(), s.A.data());
            post = s;  // closing halves on a copy: the state Alg. 1 shows the monitors (and the caller)
            mvs_kick(post, hh);
            mvs_linear_drift(post, m.data(), hh);
            t += h;
            ++k;
            from_dh<R>(post, m.data(), xm.data(), nullptr);
            const int mon = monitors(n, xm.data(), r_close, r_eject);
            if (mon != ST_ACTIVE) { st = mon; break; }
            if (!time_left(dt, (double)t, t_end) || k >= max_steps) continue;  // the loop head ends the run: no merge
            mvs_kick(s, h);                      // K(h/2) of this step + K(h/2) of the next
            mvs_linear_drift(s, m.data(), h);    // D(h/2) of this step + D(h/2) of the next (drift velocity after the kick)
        }
        if (k > 0) s = post;
        from_dh(s, m.data(), x.data(), v.data());
        for (int q = 0; q < 3 * n; ++q) { pos[q] = (double)x[q]; vel[q] = (double)v[q]; }
        *time = (double)t;
        *status = st;
        *nsteps += k;
        return;
    }
    R htrial = h;       // integrator 6: the per-system trial step, started at dt by every call
    int64_t nrej = 0;
    while (true) {
        if (!time_left(dt, (double)t, t_end)) { st = ST_DONE_TIME; break; }
        if (k >= max_steps) { st = ST_DONE_STEPS; break; }
        const R* xmon;
        R hs = h;  // the step actually taken (t += hs below)
        if (integrator == 6) {  // adaptive Runge-Kutta Cash-Karp: trial steps until one is accepted
            bool ok = false;
            bool underflow = false;
            while (true) {
                hs = htrial;
                rkck_adaptive_trial(n, x.data(), v.data(), m.data(), htrial, (R)rk_eps, &ok);
                if (ok) break;
                ++nrej;
                if (t + htrial == t) { underflow = true; break; }  // the step can no longer advance the time
            }
            if (underflow) { st = ST_STOP_STEPSIZE; break; }
            xmon = x.data();
        } else if (integrator == 0) {
            hermite_step(n, x.data(), v.data(), m.data(), h, n_corr);
            xmon = x.data();
        } else if (integrator == 4) {  // fixed-step Runge-Kutta Cash-Karp
            rkck_step(n, x.data(), v.data(), m.data(), h);
            xmon = x.data();
        } else if (integrator == 3) {  // Alg. 2 as printed: 2 evaluations per step, (a, j) carried
            hermite_step_carry(n, x.data(), v.data(), m.data(), h, ca.data(), cj.data());
            xmon = x.data();
        } else if (integrator == 2) {  // adaptive Hermite: dt is the step size scale tau of Eq. 5
            hs = hermite_adaptive_dt(n, x.data(), v.data(), m.data(), h);
            hermite_step(n, x.data(), v.data(), m.data(), hs, n_corr);
            xmon = x.data();
        } else {
            mvs_step(s, m.data(), h);
            from_dh<R>(s, m.data(), xm.data(), nullptr);
            xmon = xm.data();
        }
        t += hs;
        ++k;
        const int mon = monitors(n, xmon, r_close, r_eject);
        if (mon != ST_ACTIVE) { st = mon; break; }
    }
    if (integrator == 1) from_dh(s, m.data(), x.data(), v.data());
    for (int q = 0; q < 3 * n; ++q) { pos[q] = (double)x[q]; vel[q] = (double)v[q]; }
    *time = (double)t;
    *status = st;
    *nsteps += k;
    if (nreject) *nreject += nrej;
}

}  // namespace

// ===================================================================================================
// C interface (ctypes).  prec: 0 = double, 1 = long double.  All return 0 on success, -1 on bad arguments.
// ===================================================================================================
extern "C" {

int orc_acc_jerk(int n, const double* x, const double* v, const double* m, double* a, double* j, int prec) {
    if (n < 2 || !x || !v || !m || !a || !j) return -1;
    if (prec == 0) {
        eval_acc_jerk<double>(n, x, v, m, a, j);
    } else {
        std::vector<long double> X(x, x + 3 * n), V(v, v + 3 * n), M(m, m + n), A(3 * n), J(3 * n);
        eval_acc_jerk<long double>(n, X.data(), V.data(), M.data(), A.data(), J.data());
        for (int q = 0; q < 3 * n; ++q) { a[q] = (double)A[q]; j[q] = (double)J[q]; }
    }
    return 0;
}

// n_corr corrector iterations (the method uses 2; other values exist only for the R5b identity test)
int orc_hermite_step(int n, double* x, double* v, const double* m, double h, int n_corr, int prec) {
    if (n < 2 || !x || !v || !m) return -1;
    if (prec == 0) {
        hermite_step<double>(n, x, v, m, h, n_corr);
    } else {
        std::vector<long double> X(x, x + 3 * n), V(v, v + 3 * n), M(m, m + n);
        hermite_step<long double>(n, X.data(), V.data(), M.data(), (long double)h, n_corr);
        for (int q = 0; q < 3 * n; ++q) { x[q] = (double)X[q]; v[q] = (double)V[q]; }
    }
    return 0;
}

// integrator: 0 = Hermite (fixed step dt), 1 = MVS, 2 = adaptive Hermite (dt = tau of Eq. 5),
// 3 = Hermite with 2 evaluations per step (Alg. 2 as printed; a, j carried from step to step),
// 4 = fixed-step Runge-Kutta Cash-Karp (fifth-order solution propagated).  status/nsteps/time are in-out ([n_sys]); status STOP_* is sticky.
// 5 = MVS with merged half sub-steps, 6 = adaptive Runge-Kutta Cash-Karp (dt = first trial step, rk_eps = accuracy
// parameter; nreject [n_sys] in-out or NULL receives the rejected trial steps).
int orc_integrate2(int integrator, int64_t n_sys, int n, double* pos, double* vel, const double* mass, double* time,
                   int32_t* status, int64_t* nsteps, double dt, double t_end, int64_t max_steps, double r_close,
                   double r_eject, int prec, int nthreads, double rk_eps, int64_t* nreject) {
    if (n_sys < 0 || n < 2 || !pos || !vel || !mass || !time || !status || !nsteps) return -1;
    if (!(dt != 0) || !std::isfinite(dt) || max_steps < 0 || (integrator < 0 || integrator > 6)) return -1;
    if (integrator == 6 && !(rk_eps > 0)) return -1;
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(dynamic, 16) num_threads(nthreads)
    for (int64_t s = 0; s < n_sys; ++s) {
        double* p = pos + s * 3 * n;
        double* w = vel + s * 3 * n;
        const double* mm = mass + s * n;
        int64_t* nr = nreject ? nreject + s : nullptr;
        if (prec == 0)
            run_system<double>(integrator, n, p, w, mm, time + s, status + s, nsteps + s, dt, t_end, max_steps, r_close, r_eject, 2, rk_eps, nr);
        else
            run_system<long double>(integrator, n, p, w, mm, time + s, status + s, nsteps + s, dt, t_end, max_steps, r_close, r_eject, 2, rk_eps, nr);
    }
    return 0;
}

int orc_integrate(int integrator, int64_t n_sys, int n, double* pos, double* vel, const double* mass, double* time,
                  int32_t* status, int64_t* nsteps, double dt, double t_end, int64_t max_steps, double r_close,
                  double r_eject, int prec, int nthreads) {
    if (integrator < 0 || integrator > 4) return -1;
    return orc_integrate2(integrator, n_sys, n, pos, vel, mass, time, status, nsteps, dt, t_end, max_steps, r_close,
                          r_eject, prec, nthreads, 1e-9, nullptr);
}

// one trial step of the adaptive Cash-Karp integrator on one system (test hook): x, v, *h in-out; *r = error level,
// *accepted = 1 if the step was taken (then x, v hold the new state and *h the next trial step)
int orc_rkck_adaptive_trial(int n, double* x, double* v, const double* m, double* h, double eps, double* r, int* accepted,
                            int prec) {
    if (n < 2 || !x || !v || !m || !h || !r || !accepted || !(eps > 0)) return -1;
    bool ok = false;
    if (prec == 0) {
        *r = rkck_adaptive_trial<double>(n, x, v, m, *h, eps, &ok);
    } else {
        std::vector<long double> X(x, x + 3 * n), V(v, v + 3 * n), M(m, m + n);
        long double H = *h;
        *r = (double)rkck_adaptive_trial<long double>(n, X.data(), V.data(), M.data(), H, (long double)eps, &ok);
        for (int q = 0; q < 3 * n; ++q) { x[q] = (double)X[q]; v[q] = (double)V[q]; }
        *h = (double)H;
    }
    *accepted = ok ? 1 : 0;
    return 0;
}

// one Cash-Karp step of one system (test hook); errx, errv receive the embedded error estimate y5 - y4
int orc_rkck_step(int n, double* x, double* v, const double* m, double h, double* errx, double* errv, int prec) {
    if (n < 2 || !x || !v || !m || !errx || !errv) return -1;
    if (prec == 0) {
        rkck_step<double>(n, x, v, m, h, errx, errv);
    } else {
        std::vector<long double> X(x, x + 3 * n), V(v, v + 3 * n), M(m, m + n), EX(3 * n), EV(3 * n);
        rkck_step<long double>(n, X.data(), V.data(), M.data(), (long double)h, EX.data(), EV.data());
        for (int q = 0; q < 3 * n; ++q) { x[q] = (double)X[q]; v[q] = (double)V[q]; errx[q] = (double)EX[q]; errv[q] = (double)EV[q]; }
    }
    return 0;
}

// the Cash-Karp tableau as the oracle holds it (test hook): c[6], a[6][5] row-major, b5[6], b4[6]
int orc_rkck_tableau(double* c, double* a, double* b5, double* b4) {
    if (!c || !a || !b5 || !b4) return -1;
    const CashKarp<long double> T;
    for (int i = 0; i < 6; ++i) {
        c[i] = (double)T.c[i]; b5[i] = (double)T.b5[i]; b4[i] = (double)T.b4[i];
        for (int k = 0; k < 5; ++k) a[5 * i + k] = (double)T.a[i][k];
    }
    return 0;
}

// dt of Eq. 5 for one system (test hook)
int orc_adaptive_dt(int n, const double* x, const double* v, const double* m, double tau, double* dt, int prec) {
    if (n < 2 || !x || !v || !m || !dt) return -1;
    if (prec == 0) {
        *dt = hermite_adaptive_dt<double>(n, x, v, m, tau);
    } else {
        std::vector<long double> X(x, x + 3 * n), V(v, v + 3 * n), M(m, m + n);
        *dt = (double)hermite_adaptive_dt<long double>(n, X.data(), V.data(), M.data(), (long double)tau);
    }
    return 0;
}

int orc_energy(int64_t n_sys, int n, const double* pos, const double* vel, const double* mass, double* E, double* L, int prec) {
    if (n_sys < 0 || n < 1 || !pos || !vel || !mass || !E) return -1;
    for (int64_t s = 0; s < n_sys; ++s) {
        if (prec == 0) {
            energy_L<double>(n, pos + s * 3 * n, vel + s * 3 * n, mass + s * n, E + s, L ? L + 3 * s : nullptr);
        } else {
            std::vector<long double> X(pos + s * 3 * n, pos + (s + 1) * 3 * n), V(vel + s * 3 * n, vel + (s + 1) * 3 * n),
                M(mass + s * n, mass + (s + 1) * n);
            long double e, l[3];
            energy_L<long double>(n, X.data(), V.data(), M.data(), &e, l);
            E[s] = (double)e;
            if (L) for (int c = 0; c < 3; ++c) L[3 * s + c] = (double)l[c];
        }
    }
    return 0;
}

int orc_stumpff(double z, double* c, int prec) {
    if (!c) return -1;
    if (prec == 0) {
        stumpff<double>(z, c);
    } else {
        long double C[4];
        stumpff<long double>((long double)z, C);
        for (int q = 0; q < 4; ++q) c[q] = (double)C[q];
    }
    return 0;
}

// q, p: [3] in-out.  *iters receives the Newton iteration count (negative: bisection fallback used).
int orc_kepler_drift(double* q, double* p, double mu, double tau, int prec, int* iters) {
    if (!q || !p) return -1;
    int it;
    if (prec == 0) {
        it = kepler_drift<double>(q, p, mu, tau);
    } else {
        long double Q[3] = {q[0], q[1], q[2]}, P[3] = {p[0], p[1], p[2]};
        it = kepler_drift<long double>(Q, P, (long double)mu, (long double)tau);
        for (int c = 0; c < 3; ++c) { q[c] = (double)Q[c]; p[c] = (double)P[c]; }
    }
    if (iters) *iters = it;
    return 0;
}

// inertial Cartesian -> democratic heliocentric -> inertial Cartesian (for the coordinate round-trip test);
// Q, V out: [n][3] with row 0 = X_cm / V_cm.
int orc_dh_roundtrip(int n, const double* x, const double* v, const double* m, double* Q, double* V, double* x2, double* v2) {
    if (n < 2) return -1;
    DH<double> s;
    to_dh<double>(n, x, v, m, s);
    for (int c = 0; c < 3; ++c) { Q[c] = s.Xcm[c]; V[c] = s.Vcm[c]; }
    for (int q = 3; q < 3 * n; ++q) { Q[q] = s.Q[q]; V[q] = s.V[q]; }
    from_dh<double>(s, m, x2, v2);
    return 0;
}

}  // extern "C"
