// rkck_kernel.cuh — fused fixed-step Runge-Kutta Cash-Karp step loop for sm_100a (FP64 CUDA cores).
//
// One launch = Alg. 1 with the propagator of P:L93-97 / P:L246-248: the explicit six-stage Cash-Karp
// pair applied to y = (x, v), y' = (v, a(x)); accelerations only (Eq. 1), six evaluations per step, the
// fifth-order solution propagated (reading R-RK1).  The paper found its local variables spilling out of Fermi's
// registers and L1; here the five stored stage accelerations of a 3-body system are 90 of 255 registers.
//
// Stage velocities are never formed: with k_l = a(x_l) the stage accelerations,
//   x_i   = x + c_i h v + h^2 sum_{l <= i-2} (A A)_il k_l            (A the strictly lower tableau, c its row sums)
//   x_new = x + h v + h^2 sum_l (b A)_l k_l ,   v_new = v + h sum_i b_i k_i
// so a step is 6 evaluations and 25 DFMA per coordinate; the products c_i h, h^2 (A A)_il, h^2 (b A)_l, h b_i come
// precomputed in RkCoef (constant-bank operands).  Algebraically the oracle's formulas; rounding differs.
//
// The first evaluation of step k+1 is taken at the post-step-k positions, so its minimum pair distance is the
// close-approach monitor (as in the Hermite kernel).  Work split, pair schedule and state layout as in the Hermite
// and MVS kernels (L lanes per system, B bodies per lane; the pair evaluation is acc_pairs.cuh's acceleration-only ring
// over all N bodies).
#pragma once
#include <type_traits>
#include "acc_pairs.cuh"

namespace ensd {

struct RkCoef {
    double ch[6];       // c_i h
    double h2AA[6][4];  // h^2 (A A)_il, l = 0..i-2
    double h2bA[5];     // h^2 (b A)_l
    double hb[6];       // h b_i (fifth-order weights)
};

// ROLLED = true: stages 2 .. 6 are a loop around ONE copy of the evaluation, the stage accelerations live in local memory
// (L1-resident; they are read back once per later stage) and only the current one is in registers.  For shapes whose
// stage accelerations do not fit the registers anyway and whose straight-line step (six copies of the evaluation) no
// longer fits the instruction cache: n_body = 7, one system per thread (48 KB of code, 1.3 instruction-fetch stalls
// per issued instruction).  Same arithmetic in the same order.
template <int N, int L, int B, int MAXREG, bool ROLLED = false>
__global__ void __maxnreg__(MAXREG) rkck_kernel(View e, StepArgs p, RkCoef q) {
    constexpr int S = 32 / L;
    constexpr bool PADDED = (L * B != N);
    const int lane = threadIdx.x & 31;
    const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int sl = lane / L;
    const int l = lane - sl * L;
    const int base = sl * L;
    const int64_t sys = warp * S + sl;
    const bool live = (sl < S) && (sys < e.n_sys);
    extern __shared__ double2 ring_smem[];  // acc_ring_smem_words<L, B>() per warp (nothing for L = 1)
    double2* const W = ring_smem + (threadIdx.x >> 5) * acc_ring_smem_words<L, B>();

    double X[B][3], V[B][3], m[B];
    // time folded with the direction of the run (ts = t forward, -t backward: exact), end test ts < p.te either way
    const bool fwd = p.dt > 0.0;
    double ts = 0.0;
    int st = ENS_STOP_NONFINITE;
    bool active = false;
#pragma unroll
    for (int b = 0; b < B; ++b) {
        // dummy slot (padded shapes only): massless, at rest, far from everything and from each other
        X[b][0] = 1.0e8 * (double)(l * B + b + 1);
        X[b][1] = X[b][2] = 0.0;
        V[b][0] = V[b][1] = V[b][2] = 0.0;
        m[b] = 0.0;
    }
    if (live) {
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const int gid = l * B + b;
            if (!PADDED || gid < N) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    X[b][c] = e.pos[(int64_t)(gid * 3 + c) * e.n_pad + sys];
                    V[b][c] = e.vel[(int64_t)(gid * 3 + c) * e.n_pad + sys];
                }
                m[b] = e.mass[(int64_t)gid * e.n_pad + sys];
            }
        }
        ts = fwd ? e.time[sys] : -e.time[sys];
        st = e.status[sys];
        active = st < ENS_STOP_CLOSE;  // STOP_* are sticky; DONE_* run again
    }
    const bool writeback = active;
    const double h = p.dt;
    int64_t k = 0;
    double K[5][B][3];  // stage accelerations k_1 .. k_5
    // smallest pair r^2 of stage 1: its high word (one system per thread) or its full bit pattern (acc_pairs.cuh)
    using R2 = typename std::conditional<(L > 1), u64, unsigned>::type;
    R2 r2min;

    // The systems of the warp that run enter the loop together (mask amask) and stay in it until the exact stop logic
    // retires them (hermite_kernel.cuh): one vote and one almost never taken branch per step.
    unsigned amask = __ballot_sync(0xffffffffu, active);
    if (active) {
        while (true) {
            // stage 1 at the accepted state: also the monitors' pair distances (Alg. 1: advance, then execute(M))
            eval_acc_planets<N, L, B>(X, m, K[0], r2min, l, base, amask, W);
            // One quick test per step (as in hermite_kernel.cuh): every pair this lane saw farther apart than r_close and
            // every coordinate of its bodies below r_eject / sqrt(3), both on high words (the exact decisions cannot
            // differ; non-finite values fail it), time left, steps left.  The exact monitor / stop logic runs only when
            // some lane of the warp fails it (warp-uniform, rarely taken).
            unsigned cmax = 0u;
#pragma unroll
            for (int b = 0; b < B; ++b)
#pragma unroll
                for (int c = 0; c < 3; ++c)
                    if (!PADDED || (l * B + b < N)) cmax = max(cmax, (unsigned)__double2hiint(X[b][c]) & 0x7fffffffu);
            const bool go = (r2_high_word(r2min) > (unsigned)(p.rc2_bits >> 32)) && (cmax < p.ce_hi) && (ts < p.te) &&
                            (k < p.max_steps);
            if (__builtin_expect(__ballot_sync(amask, !go) != 0u, 0)) {
                int f = (r2_exact<N, L, B>(r2min, X, l, base, amask) < p.rc2_bits) ? 1 : 0;
#pragma unroll
                for (int b = 0; b < B; ++b) {
                    const u64 db = dbits(fma(X[b][2], X[b][2], fma(X[b][1], X[b][1], X[b][0] * X[b][0])));
                    if (!PADDED || (l * B + b < N)) {
                        if (db > p.re2_bits) f |= 2;
                        if (db > 0x7FEFFFFFFFFFFFFFull) f |= 4;  // +inf or NaN
                    }
                }
                if constexpr (L > 1) {
                    int g = f;
#pragma unroll
                    for (int i = 1; i < L; ++i) {
                        int li = l + i;
                        if (li >= L) li -= L;
                        g |= __shfl_sync(amask, f, base + li);
                    }
                    f = g;
                }
                if (k > 0 && f) {
                    st = (f & 4) ? ENS_STOP_NONFINITE : (f & 1) ? ENS_STOP_CLOSE : ENS_STOP_EJECT;
                    active = false;
                }
                if (active) {
                    if (!(ts < p.te)) {
                        st = ENS_DONE_TIME;
                        active = false;
                    } else if (k >= p.max_steps) {
                        st = ENS_DONE_STEPS;
                        active = false;
                    }
                }
                amask = __ballot_sync(amask, active);  // the lanes that go on
                if (!active) break;
            }
            if constexpr (ROLLED) {
                const unsigned am2 = amask;
                double Xs[B][3], Kt[B][3];
                double KL[6][B][3];  // k_1 .. k_6, indexed by the stage counter: local memory
                R2 dummy;
#pragma unroll
                for (int b = 0; b < B; ++b)
#pragma unroll
                    for (int c = 0; c < 3; ++c) KL[0][b][c] = K[0][b][c];
#pragma unroll 1
                for (int i = 1; i < 6; ++i) {  // stages 2 .. 6
                    const double chi = q.ch[i];
#pragma unroll
                    for (int b = 0; b < B; ++b)
#pragma unroll
                        for (int c = 0; c < 3; ++c) Xs[b][c] = fma(chi, V[b][c], X[b][c]);
#pragma unroll 1
                    for (int ll = 0; ll + 2 <= i; ++ll) {
                        const double cf = q.h2AA[i][ll];
#pragma unroll
                        for (int b = 0; b < B; ++b)
#pragma unroll
                            for (int c = 0; c < 3; ++c) Xs[b][c] = fma(cf, KL[ll][b][c], Xs[b][c]);
                    }
                    eval_acc_planets<N, L, B>(Xs, m, Kt, dummy, l, base, am2, W);
#pragma unroll
                    for (int b = 0; b < B; ++b)
#pragma unroll
                        for (int c = 0; c < 3; ++c) KL[i][b][c] = Kt[b][c];
                }
#pragma unroll
                for (int b = 0; b < B; ++b)
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        double s = fma(h, V[b][c], X[b][c]);
#pragma unroll
                        for (int ll = 0; ll < 5; ++ll) s = fma(q.h2bA[ll], KL[ll][b][c], s);
                        X[b][c] = s;
                        double w = fma(q.hb[0], KL[0][b][c], V[b][c]);  // b_2 = b_5 = 0
                        w = fma(q.hb[2], KL[2][b][c], w);
                        w = fma(q.hb[3], KL[3][b][c], w);
                        V[b][c] = fma(q.hb[5], Kt[b][c], w);
                    }
            } else {
                const unsigned am2 = amask;
                double Xs[B][3], K6[B][3];
                R2 dummy;
#pragma unroll
                for (int i = 1; i < 6; ++i) {  // stages 2 .. 6
#pragma unroll
                    for (int b = 0; b < B; ++b)
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            double s = fma(q.ch[i], V[b][c], X[b][c]);
#pragma unroll
                            for (int ll = 0; ll + 2 <= i; ++ll) s = fma(q.h2AA[i][ll], K[ll][b][c], s);
                            Xs[b][c] = s;
                        }
                    if (i < 5)
                        eval_acc_planets<N, L, B>(Xs, m, K[i], dummy, l, base, am2, W);
                    else
                        eval_acc_planets<N, L, B>(Xs, m, K6, dummy, l, base, am2, W);
                }
#pragma unroll
                for (int b = 0; b < B; ++b)
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        double s = fma(h, V[b][c], X[b][c]);
#pragma unroll
                        for (int ll = 0; ll < 5; ++ll) s = fma(q.h2bA[ll], K[ll][b][c], s);
                        X[b][c] = s;
                        double w = fma(q.hb[0], K[0][b][c], V[b][c]);  // b_2 = b_5 = 0
                        w = fma(q.hb[2], K[2][b][c], w);
                        w = fma(q.hb[3], K[3][b][c], w);
                        V[b][c] = fma(q.hb[5], K6[b][c], w);
                    }
            }
            ts += fabs(h);
            ++k;
        }
    }

    if (writeback) {
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const int gid = l * B + b;
            if (!PADDED || gid < N) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    e.pos[(int64_t)(gid * 3 + c) * e.n_pad + sys] = X[b][c];
                    e.vel[(int64_t)(gid * 3 + c) * e.n_pad + sys] = V[b][c];
                }
            }
        }
        if (l == 0) {
            e.time[sys] = fwd ? ts : -ts;
            e.status[sys] = st;
            e.nsteps[sys] += k;
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Adaptive-step Cash-Karp (reading R-RK2' of DESIGN.md section 3: the step-size control the GSL
// manual documents for the stepper the paper follows, step factors from a discrete set).  Per system and trial step h:
//   error level  r = max( max|err_x| / (eps X), max|err_v| / (eps V) ),  err = fifth minus fourth order solution,
//                X = max_b |x_b|, V = max_b |v_b| at the start of the step;
//   r > 1.1      rejected: state and time untouched, h <- h max(1/5, F(0.9 r^(-1/4))), next trial;
//   otherwise    accepted; if r < 0.5 the next step starts from h <- h min(5, max(1, F(0.9 r^(-1/5))));  F(f) = floor(16 f) / 16.
// With k_l the stage accelerations and d = b5 - b4 (sum d_i = 0) the error needs no stage velocities either:
//   err_x = h^2 sum_l (d A)_l k_l,   err_v = h sum_i d_i k_i.
// The step size is per system, so the tableau products come without the powers of h (RkUnit, constant bank) and h, h^2
// multiply the sums.  Stage 1 depends on the positions only: a rejected trial keeps it (bit-identical to re-evaluating).
// Systems take different numbers of trials, so the grid is persistent and every group of L lanes pulls the next system
// from a device counter when its own is finished (as the adaptive Hermite kernel does).
// ---------------------------------------------------------------------------------------------------------------
struct RkUnit {
    double c[6];       // c_i
    double AA[6][4];   // (A A)_il
    double bA[5];      // (b5 A)_l
    double b[6];       // b5_i
    double dA[5];      // ((b5 - b4) A)_l
    double d[6];       // b5_i - b4_i
};

// r^(-1/5) for 1e-4 <= r < 0.5: FP32 seed (exp2 / log2 approximations, ~1e-6) and two Newton steps for y^-5 = r
__device__ __forceinline__ double inv_fifth_root(double r) {
    double y = (double)exp2f(-0.2f * __log2f((float)r));
#pragma unroll
    for (int it = 0; it < 2; ++it) {
        const double y2 = y * y, y5 = (y2 * y2) * y;
        y = fma(0.2 * y, fma(-r, y5, 1.0), y);
    }
    return y;
}

template <int N, int L, int B, int MAXREG, bool ROLLED = false>
__global__ void __maxnreg__(MAXREG) rkck_adaptive_kernel(View e, StepArgs p, RkUnit q) {
    constexpr int S = 32 / L;
    constexpr bool PADDED = (L * B != N);
    const int lane = threadIdx.x & 31;
    const int sl = lane / L;
    const int l = lane - sl * L;
    const int base = sl * L;
    int64_t sys = 0;
    extern __shared__ double2 ring_smem[];  // acc_ring_smem_words<L, B>() per warp (nothing for L = 1)
    double2* const W = ring_smem + (threadIdx.x >> 5) * acc_ring_smem_words<L, B>();

    double X[B][3], V[B][3], m[B];
    double t = 0.0, h = p.dt;
    int st = ENS_STOP_NONFINITE;
    bool active = false, writeback = false, have_k1 = false;
    int64_t k = 0, nrej = 0;
    bool exhausted = !(sl < S);
    const bool fwd = p.dt > 0.0;
    const double ieps = 1.0 / p.rk_eps;

    auto load_system = [&]() {
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const int gid = l * B + b;
            X[b][0] = 1.0e8 * (double)(gid + 1);  // dummy slot (padded shapes): massless, far from everything
            X[b][1] = X[b][2] = 0.0;
            V[b][0] = V[b][1] = V[b][2] = 0.0;
            m[b] = 0.0;
            if (!PADDED || gid < N) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    X[b][c] = e.pos[(int64_t)(gid * 3 + c) * e.n_pad + sys];
                    V[b][c] = e.vel[(int64_t)(gid * 3 + c) * e.n_pad + sys];
                }
                m[b] = e.mass[(int64_t)gid * e.n_pad + sys];
            }
        }
        t = e.time[sys];
        st = e.status[sys];
        k = nrej = 0;
        h = p.dt;  // every call starts every system from the caller's trial step
        have_k1 = false;
        active = st < ENS_STOP_CLOSE;
        writeback = active;
    };
    auto store_system = [&]() {
        if (writeback) {
#pragma unroll
            for (int b = 0; b < B; ++b) {
                const int gid = l * B + b;
                if (!PADDED || gid < N) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        e.pos[(int64_t)(gid * 3 + c) * e.n_pad + sys] = X[b][c];
                        e.vel[(int64_t)(gid * 3 + c) * e.n_pad + sys] = V[b][c];
                    }
                }
            }
            if (l == 0) {
                e.time[sys] = t;
                e.status[sys] = st;
                e.nsteps[sys] += k;
                e.nreject[sys] += nrej;
            }
        }
        writeback = false;
    };
    auto refill = [&]() -> bool {  // whole warp converged
        const bool want = !active && !exhausted;
        const unsigned rmask = __ballot_sync(0xffffffffu, want);
        if (want) {
            store_system();
            unsigned long long idx = 0;
            if (l == 0) idx = atomicAdd(p.counter, 1ull);
            if constexpr (L > 1) idx = __shfl_sync(rmask, idx, base);
            if ((int64_t)idx < e.n_sys) {
                sys = p.order ? (int64_t)p.order[idx] : (int64_t)idx;  // longest expected run first (adaptive_order.cu)
                load_system();
            } else {
                exhausted = true;
            }
        }
        return __ballot_sync(0xffffffffu, !exhausted) != 0;
    };
    // maximum over the L lanes of a system (all lanes of `mask` systems take part)
    auto lanes_max = [&](double v, unsigned mask) {
        if constexpr (L > 1) {
            double g = v;
#pragma unroll
            for (int i = 1; i < L; ++i) {
                int li = l + i;
                if (li >= L) li -= L;
                g = fmax(g, __shfl_sync(mask, v, base + li));
            }
            return g;
        } else {
            return v;
        }
    };

    double K[5][B][3];  // stage accelerations k_1 .. k_5
    // smallest pair r^2 of stage 1: its high word (one system per thread) or its full bit pattern (acc_pairs.cuh)
    using R2 = typename std::conditional<(L > 1), u64, unsigned>::type;
    R2 r2min;

    while (true) {
        if (!refill()) break;
        const unsigned amask = __ballot_sync(0xffffffffu, active);
        if (amask == 0) continue;
        if (active) {
            // stage 1 at the accepted state (after an accepted step or at the start of the run): also the monitors'
            // pair distances (Alg. 1: advance, then execute(M)) and the loop tests.  A rejected trial skips all this.
            const unsigned kmask = __ballot_sync(amask, !have_k1);  // the lanes that take stage 1 (and its quick test)
            if (!have_k1) {
                eval_acc_planets<N, L, B>(X, m, K[0], r2min, l, base, kmask, W);
                have_k1 = true;
                // the quick test of the fixed-step kernel; the exact logic only when some lane of kmask fails it
                unsigned cmax = 0u;
#pragma unroll
                for (int b = 0; b < B; ++b)
#pragma unroll
                    for (int c = 0; c < 3; ++c)
                        if (!PADDED || (l * B + b < N)) cmax = max(cmax, (unsigned)__double2hiint(X[b][c]) & 0x7fffffffu);
                const bool go = (r2_high_word(r2min) > (unsigned)(p.rc2_bits >> 32)) && (cmax < p.ce_hi) &&
                                (fwd ? (t < p.t_end) : (t > p.t_end)) && (k < p.max_steps);
                if (__builtin_expect(__ballot_sync(kmask, !go) != 0u, 0)) {
                    int f = (r2_exact<N, L, B>(r2min, X, l, base, kmask) < p.rc2_bits) ? 1 : 0;
#pragma unroll
                    for (int b = 0; b < B; ++b) {
                        const u64 db = dbits(fma(X[b][2], X[b][2], fma(X[b][1], X[b][1], X[b][0] * X[b][0])));
                        if (!PADDED || (l * B + b < N)) {
                            if (db > p.re2_bits) f |= 2;
                            if (db > 0x7FEFFFFFFFFFFFFFull) f |= 4;
                        }
                    }
                    if constexpr (L > 1) {
                        int g = f;
#pragma unroll
                        for (int i = 1; i < L; ++i) {
                            int li = l + i;
                            if (li >= L) li -= L;
                            g |= __shfl_sync(kmask, f, base + li);
                        }
                        f = g;
                    }
                    if (k > 0 && f) {
                        st = (f & 4) ? ENS_STOP_NONFINITE : (f & 1) ? ENS_STOP_CLOSE : ENS_STOP_EJECT;
                        active = false;
                    } else if (!(fwd ? (t < p.t_end) : (t > p.t_end))) {
                        st = ENS_DONE_TIME;
                        active = false;
                    } else if (k >= p.max_steps) {
                        st = ENS_DONE_STEPS;
                        active = false;
                    }
                }
            }
            unsigned am2 = amask;
            if constexpr (L > 1) am2 = __ballot_sync(amask, active);
            if (active) {
                const double h2 = h * h;
                double Xs[B][3], K6[B][3];
                double KL[ROLLED ? 6 : 1][B][3];  // ROLLED (see rkck_kernel): k_1 .. k_6 in local memory, one copy of the evaluation
                R2 dummy;
                if constexpr (ROLLED) {
#pragma unroll
                    for (int b = 0; b < B; ++b)
#pragma unroll
                        for (int c = 0; c < 3; ++c) KL[0][b][c] = K[0][b][c];
#pragma unroll 1
                    for (int i = 1; i < 6; ++i) {  // stages 2 .. 6
                        const double ch = q.c[i] * h;
                        double S[B][3];
#pragma unroll
                        for (int b = 0; b < B; ++b)
#pragma unroll
                            for (int c = 0; c < 3; ++c) S[b][c] = 0.0;
#pragma unroll 1
                        for (int ll = 0; ll + 2 <= i; ++ll) {
                            const double cf = q.AA[i][ll];
#pragma unroll
                            for (int b = 0; b < B; ++b)
#pragma unroll
                                for (int c = 0; c < 3; ++c) S[b][c] = fma(cf, KL[ll][b][c], S[b][c]);
                        }
#pragma unroll
                        for (int b = 0; b < B; ++b)
#pragma unroll
                            for (int c = 0; c < 3; ++c) Xs[b][c] = fma(h2, S[b][c], fma(ch, V[b][c], X[b][c]));
                        eval_acc_planets<N, L, B>(Xs, m, K6, dummy, l, base, am2, W);
#pragma unroll
                        for (int b = 0; b < B; ++b)
#pragma unroll
                            for (int c = 0; c < 3; ++c) KL[i][b][c] = K6[b][c];
                    }
                } else {
#pragma unroll
                    for (int i = 1; i < 6; ++i) {  // stages 2 .. 6
                        const double ch = q.c[i] * h;
#pragma unroll
                        for (int b = 0; b < B; ++b)
#pragma unroll
                            for (int c = 0; c < 3; ++c) {
                                double s = 0.0;
#pragma unroll
                                for (int ll = 0; ll + 2 <= i; ++ll) s = fma(q.AA[i][ll], K[ll][b][c], s);
                                Xs[b][c] = fma(h2, s, fma(ch, V[b][c], X[b][c]));
                            }
                        if (i < 5)
                            eval_acc_planets<N, L, B>(Xs, m, K[i], dummy, l, base, am2, W);
                        else
                            eval_acc_planets<N, L, B>(Xs, m, K6, dummy, l, base, am2, W);
                    }
                }
                // the stage accelerations the sums below read: registers, or the local-memory copy
                auto& KK = *[&] {
                    if constexpr (ROLLED) return &KL;
                    else return &K;
                }();
                // error level of this trial (scales from the state the step starts from)
                double ex = 0.0, ev = 0.0, x2 = 0.0, v2 = 0.0;
#pragma unroll
                for (int b = 0; b < B; ++b) {
                    if (!PADDED || (l * B + b < N)) {
                        x2 = fmax(x2, fma(X[b][2], X[b][2], fma(X[b][1], X[b][1], X[b][0] * X[b][0])));
                        v2 = fmax(v2, fma(V[b][2], V[b][2], fma(V[b][1], V[b][1], V[b][0] * V[b][0])));
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            double sx = 0.0;
#pragma unroll
                            for (int ll = 0; ll < 5; ++ll) sx = fma(q.dA[ll], KK[ll][b][c], sx);
                            double sv = q.d[0] * KK[0][b][c];  // d_2 = 0
                            sv = fma(q.d[2], KK[2][b][c], sv);
                            sv = fma(q.d[3], KK[3][b][c], sv);
                            sv = fma(q.d[4], KK[4][b][c], sv);
                            sv = fma(q.d[5], K6[b][c], sv);
                            ex = fmax(ex, fabs(sx));
                            ev = fmax(ev, fabs(sv));
                        }
                    }
                }
                ex = lanes_max(ex, am2) * h2;
                ev = lanes_max(ev, am2) * fabs(h);
                x2 = lanes_max(x2, am2);
                v2 = lanes_max(v2, am2);
                // r = max(ex / (eps |x|), ev / (eps |v|)); NaN (a broken state) compares false everywhere: accepted, and
                // the non-finite monitor stops the system at its next stage 1
                const double rx = (ex * ieps) * rsqrt_f64(x2), rv = (ev * ieps) * rsqrt_f64(v2);
                const double r = rx > rv ? rx : rv;
                if (r > 1.1) {
                    double f = 0.2;
                    if (r < 1e300) {
                        const double g = rsqrt_f64(r * rsqrt_f64(r));  // r^(-1/4)
                        f = floor(16.0 * (0.9 * g)) * 0.0625;
                        if (!(f >= 0.2)) f = 0.2;
                    }
                    h *= f;
                    ++nrej;
                    if (t + h == t) {  // the step no longer advances the time
                        st = ENS_STOP_STEPSIZE;
                        active = false;
                    }
                } else {
#pragma unroll
                    for (int b = 0; b < B; ++b)
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            double s = 0.0;
#pragma unroll
                            for (int ll = 0; ll < 5; ++ll) s = fma(q.bA[ll], KK[ll][b][c], s);
                            X[b][c] = fma(h2, s, fma(h, V[b][c], X[b][c]));
                            double w = q.b[0] * KK[0][b][c];  // b_2 = b_5 = 0
                            w = fma(q.b[2], KK[2][b][c], w);
                            w = fma(q.b[3], KK[3][b][c], w);
                            w = fma(q.b[5], K6[b][c], w);
                            V[b][c] = fma(h, w, V[b][c]);
                        }
                    t += h;
                    ++k;
                    have_k1 = false;
                    if (r < 0.5) {
                        double f = 5.0;
                        if (r >= 1e-4) {
                            f = floor(16.0 * (0.9 * inv_fifth_root(r))) * 0.0625;
                            f = f > 5.0 ? 5.0 : f < 1.0 ? 1.0 : f;
                        }
                        h *= f;
                    }
                }
            }
        }
    }
    store_system();
}

}  // namespace ensd
