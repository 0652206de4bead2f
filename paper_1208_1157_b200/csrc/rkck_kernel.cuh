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
#include "acc_pairs.cuh"

namespace ensd {

struct RkCoef {
    double ch[6];       // c_i h
    double h2AA[6][4];  // h^2 (A A)_il, l = 0..i-2
    double h2bA[5];     // h^2 (b A)_l
    double hb[6];       // h b_i (fifth-order weights)
};

template <int N, int L, int B, int MAXREG>
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

    double X[B][3], V[B][3], m[B];
    double t = 0.0;
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
        t = e.time[sys];
        st = e.status[sys];
        active = st < ENS_STOP_CLOSE;  // STOP_* are sticky; DONE_* run again
    }
    const bool writeback = active;
    const double h = p.dt;
    const bool fwd = h > 0.0;
    int64_t k = 0;
    double K[5][B][3];  // stage accelerations k_1 .. k_5
    u64 r2min;

    while (true) {
        const unsigned amask = __ballot_sync(0xffffffffu, active);
        if (amask == 0) break;
        if (active) {
            // stage 1 at the accepted state: also the monitors' pair distances (Alg. 1: advance, then execute(M))
            eval_acc_planets<N, L, B>(X, m, K[0], r2min, l, base, amask);
            {
                constexpr bool PADDED2 = PADDED;
                int f = (r2min < p.rc2_bits) ? 1 : 0;
#pragma unroll
                for (int b = 0; b < B; ++b) {
                    const u64 db = dbits(fma(X[b][2], X[b][2], fma(X[b][1], X[b][1], X[b][0] * X[b][0])));
                    if (!PADDED2 || (l * B + b < N)) {
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
            }
            if (active) {
                if (!(fwd ? (t < p.t_end) : (t > p.t_end))) {
                    st = ENS_DONE_TIME;
                    active = false;
                } else if (k >= p.max_steps) {
                    st = ENS_DONE_STEPS;
                    active = false;
                }
            }
            // lanes that just stopped take no part in the shuffles of the remaining stages
            unsigned am2 = amask;
            if constexpr (L > 1) am2 = __ballot_sync(amask, active);
            if (active) {
                double Xs[B][3], K6[B][3];
                u64 dummy;
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
                        eval_acc_planets<N, L, B>(Xs, m, K[i], dummy, l, base, am2);
                    else
                        eval_acc_planets<N, L, B>(Xs, m, K6, dummy, l, base, am2);
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
                t += h;
                ++k;
            }
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
            e.time[sys] = t;
            e.status[sys] = st;
            e.nsteps[sys] += k;
        }
    }
}

}  // namespace ensd
