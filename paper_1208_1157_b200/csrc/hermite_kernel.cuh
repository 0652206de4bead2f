// hermite_kernel.cuh — the fused Hermite step loop for sm_100a (FP64 CUDA cores; no tensor cores: not a contraction).
//
// One launch = Alg. 1 for every system: state is read from the SoA rows once, lives in registers
// for all steps and is written back once.  One step = Alg. 2: predictor (Eq. 3,
// P:L79-81), then two corrector iterations (Eq. 4, read as R3-R5 of DESIGN.md §3), each preceded by an
// acceleration-and-jerk evaluation (Eq. 1; jerk P:L77) — 3 evaluations per step (R6).
//
// Work split (differs from the paper's Fermi design): a system is held by L lanes of a warp (L odd),
// B bodies per lane.  Every unordered pair is evaluated exactly once:
//   * pairs of two bodies of the same lane: in registers;
//   * pairs across lanes: ring schedule.  At shift s = 1..(L-1)/2 lane l is visited by the bodies of lane (l+s) mod L
//     (read from the warp's own shared memory, where every lane publishes its bodies once per evaluation),
//     accumulates its own half of each pair in registers and the visitor's half (Newton's third law) in a temporary
//     that goes back to the owner by shuffle or through the owner's shared-memory slot.  No __syncthreads.
// L = 1 (n_body <= 8) is "one system per thread" and touches neither shared memory nor shuffles.
//
// The first evaluation of step k+1 is the evaluation of the post-step-k state, so its minimum pair distance IS
// the close-approach monitor Alg. 1 places after step k: monitors cost no extra pair work, and a
// launch costs 3 evaluations per step + 1.  The monitors and the loop tests are one quick test per step on high words
// (integer ALU) and one vote; the exact logic runs behind a warp-uniform, rarely taken branch (quick_test, exact_stop).
// A system that stops (monitor, t_end, step budget) leaves the step loop; the other systems of the warp go on under
// the reduced mask and the warp is done when none is left, so finished systems consume no FP64 issue slots
// (north_star item 3).
#pragma once
#include "ens_device.cuh"

namespace ensd {

// One unordered pair (i, k): adds m_k f to (a_i, j_i) and -m_i f to (a_k, j_k), with
//   f_a = dx / r^3,  f_j = (dv - 3 (dx.dv) dx / r^2) / r^3,  dx = x_k - x_i, dv = v_k - v_i   (Eq. 1 and d/dt, R1-R2).
// 38 FP64 instructions.  r2 is returned for the close-approach monitor.
// FIRST_K = true: (a_k, j_k) are assigned, not accumulated (the visitor's sums start with this pair: saves clearing them).
template <bool FIRST_K = false>
__device__ __forceinline__ double pair_acc_jerk(const double (&xi)[3], const double (&vi)[3], double mi,
                                                double (&ai)[3], double (&ji)[3], const double (&xk)[3],
                                                const double (&vk)[3], double mk, double (&ak)[3],
                                                double (&jk)[3]) {
    double dx[3], dv[3], u[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        dx[c] = xk[c] - xi[c];
        dv[c] = vk[c] - vi[c];
    }
    const double r2 = fma(dx[2], dx[2], fma(dx[1], dx[1], dx[0] * dx[0]));
    const double rv = fma(dx[2], dv[2], fma(dx[1], dv[1], dx[0] * dv[0]));
    const double y = rsqrt_f64(r2);
    const double y2 = y * y;
    const double y3 = y2 * y;
    const double s3 = (-3.0 * y2) * rv;
    const double wi = mk * y3;
    const double wk = -mi * y3;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        u[c] = fma(s3, dx[c], dv[c]);
        ai[c] = fma(wi, dx[c], ai[c]);
        ji[c] = fma(wi, u[c], ji[c]);
        if constexpr (FIRST_K) {
            ak[c] = wk * dx[c];
            jk[c] = wk * u[c];
        } else {
            ak[c] = fma(wk, dx[c], ak[c]);
            jk[c] = fma(wk, u[c], jk[c]);
        }
    }
    return r2;
}

// Shared memory of the cross-lane schedule (L > 1 only), per warp, in 16-byte words laid out word-major (word w of lane
// n at [w * 32 + n]: a warp's access touches every bank group once per quarter warp unless two systems of the quarter
// straddle it):
//   visitors  B * 4 words per lane: (x0, x1) (x2, v0) (v1, v2) (m, -) of each of the lane's bodies
//   returns   2 * 3 words per lane: (a0, a1) (a2, j0) (j1, j2), double-buffered over the visits (RET_SMEM shapes)
template <int L, int B>
__host__ __device__ constexpr int ring_smem_words() {
    return L > 1 ? B * 4 * 32 + 6 * 32 : 0;
}
// which shapes send the returned halves through shared memory instead of shuffles (measured, DESIGN.md section 8:
// a gain for 5 lanes x 3 bodies, a loss for the shapes with 2 bodies per lane, neutral for 3 lanes)
template <int L, int B>
__host__ __device__ constexpr bool ring_returns_in_smem() {
    return L == 5 && B == 3;
}

// Acceleration and jerk of the B bodies this lane owns, every pair of the system once.
// l = lane index inside the system (0..L-1), base = first lane of the system in the warp, amask = active lanes,
// W = this warp's shared memory (ring_smem_words; unused for L = 1).
// TRACK = false skips the minimum pair distance (only a step's first evaluation feeds the monitor).  The minimum is
// kept as the smallest HIGH WORD of the squared separations' bit patterns (one integer min per pair, off the FP64
// pipe); monitor_flags decides exactly from it, recomputing the full 64-bit minimum only in the rare tie.
template <int N, int L, int B, bool TRACK = true>
__device__ __forceinline__ void eval_acc_jerk(const double (&x)[B][3], const double (&v)[B][3], const double (&m)[B],
                                              double (&a)[B][3], double (&j)[B][3], unsigned& r2min, int l, int base,
                                              unsigned amask, double2* W) {
    constexpr bool PADDED = (L * B != N);
    constexpr bool RET_SMEM = ring_returns_in_smem<L, B>();
#pragma unroll
    for (int b = 0; b < B; ++b)
#pragma unroll
        for (int c = 0; c < 3; ++c) a[b][c] = j[b][c] = 0.0;
    if constexpr (TRACK) r2min = ~0u;

    // Cross-lane schedule (L > 1): every lane publishes its bodies in shared memory (four 16-byte stores per body,
    // two warp barriers per evaluation) and reads the visiting body right before the pairs that use it (four 16-byte
    // loads instead of the 14 shuffles and the double-buffered visitor registers of the earlier shuffle ring):
    //   publish | in-lane pairs among bodies 1.. |
    //   for s = 1..H, for each visitor body c: { read body c of lane l + s | B pairs (my bodies x visitor c) |
    //                                            add the returns for my body c-1 | send the returns for visitor c } |
    //   in-lane pairs with body 0 | add the last returns
    // The returned halves (Newton's third law: the visitor's share of the B pairs) travel by shuffle, or through the
    // owner's shared-memory slot where that is faster (RET_SMEM), and are added one visit behind.
    constexpr int H = (L - 1) / 2;
    const int wl = threadIdx.x & 31;
    if constexpr (L > 1) {
        __syncwarp(amask);  // every lane has finished reading the previous publication
#pragma unroll
        for (int c = 0; c < B; ++c) {
            W[(c * 4 + 0) * 32 + wl] = make_double2(x[c][0], x[c][1]);
            W[(c * 4 + 1) * 32 + wl] = make_double2(x[c][2], v[c][0]);
            W[(c * 4 + 2) * 32 + wl] = make_double2(v[c][1], v[c][2]);
            W[(c * 4 + 3) * 32 + wl] = make_double2(m[c], 0.0);
        }
        __syncwarp(amask);
    }
    double xv[3], vv[3], mv;  // the visiting body
    auto fetch_body = [&](int src, int c) {
        const double2 w0 = W[(c * 4 + 0) * 32 + src], w1 = W[(c * 4 + 1) * 32 + src], w2 = W[(c * 4 + 2) * 32 + src],
                      w3 = W[(c * 4 + 3) * 32 + src];
        xv[0] = w0.x, xv[1] = w0.y, xv[2] = w1.x;
        vv[0] = w1.y, vv[1] = w2.x, vv[2] = w2.y;
        mv = w3.x;
    };

    // pairs inside the lane.  Order: pairs among bodies 1.. first, pairs with local body 0 last, so that on lane 0
    // every planet receives the star's (largest) contribution last (for L = 1 this is exactly the
    // oracle's order: planets ascending, then the star).
    auto in_lane = [&](int b) {
#pragma unroll
        for (int c = b + 1; c < B; ++c) {
            const double r2 = pair_acc_jerk(x[b], v[b], m[b], a[b], j[b], x[c], v[c], m[c], a[c], j[c]);
            if constexpr (TRACK) min_hi(r2min, r2, !PADDED || (l * B + c < N));
        }
    };
#pragma unroll
    for (int b = 1; b < B; ++b) in_lane(b);

    if constexpr (L > 1) {
        double2* const R = W + B * 4 * 32;  // return slots
        double ra[3], rj[3];                // shuffle path: the other half of the pairs of ONE of my bodies, in flight
        auto add_returns = [&](int body, int slot) {
            if constexpr (RET_SMEM) {
                const double2 r0 = R[(slot * 3 + 0) * 32 + wl], r1 = R[(slot * 3 + 1) * 32 + wl],
                              r2 = R[(slot * 3 + 2) * 32 + wl];
                ra[0] = r0.x, ra[1] = r0.y, ra[2] = r1.x;
                rj[0] = r1.y, rj[1] = r2.x, rj[2] = r2.y;
            }
#pragma unroll
            for (int q = 0; q < 3; ++q) {
                a[body][q] += ra[q];
                j[body][q] += rj[q];
            }
        };
#pragma unroll
        for (int s = 1; s <= H; ++s) {
            int ls = l + s;  // whose bodies visit this lane at shift s: it owns the halves computed here
            if (ls >= L) ls -= L;
            int lr = l - s;  // the lane this lane's bodies visit: it computes the halves this lane gets back
            if (lr < 0) lr += L;
#pragma unroll
            for (int c = 0; c < B; ++c) {
                const int vis = (s - 1) * B + c;
                fetch_body(base + ls, c);
                double av[3], jv[3];  // the visitor's half of these B pairs: started by the first pair
                const bool vvalid = !PADDED || (ls * B + c < N);
#pragma unroll
                for (int b = 0; b < B; ++b) {
                    const double r2 = b == 0 ? pair_acc_jerk<true>(x[b], v[b], m[b], a[b], j[b], xv, vv, mv, av, jv)
                                             : pair_acc_jerk(x[b], v[b], m[b], a[b], j[b], xv, vv, mv, av, jv);
                    if constexpr (TRACK) min_hi(r2min, r2, vvalid && (!PADDED || (l * B + b < N)));
                }
                if constexpr (RET_SMEM) {
                    if (vis >= 1) {
                        __syncwarp(amask);  // the returns of the previous visit are written (and its slot's last reads done)
                        add_returns((vis - 1) % B, (vis - 1) & 1);
                    }
                    R[((vis & 1) * 3 + 0) * 32 + base + ls] = make_double2(av[0], av[1]);
                    R[((vis & 1) * 3 + 1) * 32 + base + ls] = make_double2(av[2], jv[0]);
                    R[((vis & 1) * 3 + 2) * 32 + base + ls] = make_double2(jv[1], jv[2]);
                } else {
                    if (vis >= 1) add_returns((vis - 1) % B, 0);  // sent one visit ago
#pragma unroll
                    for (int q = 0; q < 3; ++q) {
                        ra[q] = __shfl_sync(amask, av[q], base + lr);
                        rj[q] = __shfl_sync(amask, jv[q], base + lr);
                    }
                }
            }
        }
        in_lane(0);
        if constexpr (RET_SMEM) __syncwarp(amask);
        add_returns(B - 1, (H * B - 1) & 1);
    } else {
        in_lane(0);
    }
}

// Adaptive time step, Eq. 5: dt = tau [ sum_i |j_i|^2 / |a_i|^2 ]^(-1/2) over ALL bodies of the system
// (R-A1), from the acceleration and jerk at the beginning of the step; bodies that feel no acceleration are left out
// (R-A2).  Every lane of the system gathers the per-lane partial sums in the same (lane) order, so all of them take
// bit-identical steps.  Reciprocal and reciprocal square root are the seeded + refined ones of ens_device.cuh (<= 1 ulp).
template <int N, int L, int B>
__device__ __forceinline__ double adaptive_dt(const double (&a)[B][3], const double (&j)[B][3], double tau, int l,
                                              int base, unsigned amask) {
    constexpr bool PADDED = (L * B != N);
    double part = 0.0;
#pragma unroll
    for (int b = 0; b < B; ++b) {
        const double a2 = fma(a[b][2], a[b][2], fma(a[b][1], a[b][1], a[b][0] * a[b][0]));
        const double j2 = fma(j[b][2], j[b][2], fma(j[b][1], j[b][1], j[b][0] * j[b][0]));
        const double ia2 = a2 > 1e-290 ? rcp_f64<true>(a2) : 0.0;  // R-A2: no acceleration, no term
        if (!PADDED || (l * B + b < N)) part = fma(j2, ia2, part);
    }
    double sum = part;
    if constexpr (L > 1) {
        sum = __shfl_sync(amask, part, base);
#pragma unroll
        for (int i = 1; i < L; ++i) sum += __shfl_sync(amask, part, base + i);
    }
    return tau * rsqrt_f64(sum);
}

// bits: 1 = close approach, 2 = ejection, 4 = non-finite position; OR-reduced over the lanes of the system.
// r2min_hi = smallest high word of the squared pair separations this lane saw.  r^2 < r_close^2 (the exact 64-bit test,
// R11) follows from the high words alone unless the two are equal; then (only then: the minimum separation is within
// 2^-20 of the threshold) the systems concerned recompute the exact minimum from the positions, which are the ones
// the evaluation used, in the same arithmetic.
template <int N, int L, int B>
__device__ __forceinline__ int monitor_flags(const double (&x)[B][3], unsigned r2min_hi, const StepArgs& p, int l,
                                             int base, unsigned amask) {
    constexpr bool PADDED = (L * B != N);
    const unsigned rc_hi = (unsigned)(p.rc2_bits >> 32);
    int f = (r2min_hi < rc_hi) ? 1 : (r2min_hi == rc_hi) ? 8 : 0;
#pragma unroll
    for (int b = 0; b < B; ++b) {
        const double d2 = fma(x[b][2], x[b][2], fma(x[b][1], x[b][1], x[b][0] * x[b][0]));
        const u64 db = dbits(d2);
        if (!PADDED || (l * B + b < N)) {
            if (db > p.re2_bits) f |= 2;
            if (db > 0x7FEFFFFFFFFFFFFFull) f |= 4;  // > DBL_MAX: +inf or NaN
        }
    }
    auto reduce = [&](int v, unsigned mask) {
        if constexpr (L > 1) {
            int g = v;
#pragma unroll
            for (int i = 1; i < L; ++i) {
                int li = l + i;
                if (li >= L) li -= L;
                g |= __shfl_sync(mask, v, base + li);
            }
            return g;
        } else {
            return v;
        }
    };
    f = reduce(f, amask);
    const bool tie = (f & 9) == 8;  // the same for every lane of a system
    unsigned tmask = amask;
    if constexpr (L > 1) tmask = __ballot_sync(amask, tie);
    if (tie) {
        const int c = pair_r2min<N, L, B>(x, l, base, tmask) < p.rc2_bits ? 1 : 0;
        f |= reduce(c, tmask);
    }
    return f & 7;
}

// UNROLL = 1: the three evaluations of a step are three inlined copies (straight-line step, best for small pair
// counts); 2: the same with the two corrector iterations as one copy in a loop (two copies of the evaluation);
// 0: one copy of the evaluation inside a 3-phase loop (keeps large-n kernels inside the instruction cache and the
// live register set at x, v, C_x, C_v, a, j).
// ADAPT = true: the adaptive-step integrator (Eq. 5): p.dt is the step size scale tau, the step h and the ten
// coefficients are per system and per step (registers) instead of launch constants.
// CARRY = true: Alg. 2 exactly as printed (reading R6-alt): two evaluations per step; (a0, j0) of a step
// are the (a2, j2) the previous step's last evaluation left in the registers; only the first step of a launch
// evaluates at the state itself.  A third less pair work per step; the step is no longer a pure function of (x, v).
// SLICED = true (fixed step, 3 evaluations): a persistent grid that time-slices the ensemble.  The step is a pure
// function of the state (R6), so a run of max_steps steps equals ceil(max_steps / K) back-to-back runs of K steps with
// the state parked in the SoA rows (L2-resident) in between, bit for bit.  Warps pull tasks (warp-group g of S systems,
// slice s) from a device counter, slice-major, so all groups advance at the same rate and an ensemble of, say, 1.15
// waves of resident warps keeps every warp slot busy until the last slice instead of running a second, nearly empty
// wave for a whole pass (config 3: DESIGN.md section 6.1).  slice_done[g] orders slice s + 1 of a group after slice s.
template <int N, int L, int B, int UNROLL, int MAXT, int MINB, bool ADAPT = false, bool CARRY = false,
          bool SLICED = false>
__global__ void __launch_bounds__(MAXT, MINB) hermite_kernel(View e, StepArgs p) {
    static_assert(!(ADAPT && CARRY), "the carried (a, j) are not kept across refills");
    static_assert(!(SLICED && (ADAPT || CARRY)), "time slices need a step that is a pure function of the state");
    constexpr int S = 32 / L;  // systems per warp
    constexpr bool PADDED = (L * B != N);
    const int lane = threadIdx.x & 31;
    const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    extern __shared__ double2 ring_smem[];  // ring_smem_words<L, B>() per warp (nothing for L = 1)
    double2* const W = ring_smem + (threadIdx.x >> 5) * ring_smem_words<L, B>();
    const int sl = lane / L;
    const int l = lane - sl * L;
    const int base = sl * L;
    // Fixed step: system (warp * S + sl) for the whole launch.  ADAPT: a persistent grid; every group of L lanes pulls
    // system indices from a device counter and pulls the next one when its system finishes (systems take different
    // numbers of steps: a finished system must not leave its lanes idle until the slowest of the warp is done).
    int64_t sys = warp * S + sl;

    double X[B][3], V[B][3], m[B];
    // Time is kept folded with the direction of the run: ts = t going forward, -t going backward (negation is exact,
    // so ts += |h| mirrors t += h bit for bit) and the end test is the one comparison ts < p.te in both directions.
    const bool fwd = p.dt > 0.0;
    double ts = 0.0;
    int st = ENS_STOP_NONFINITE;
    bool active = false, writeback = false;
    int64_t k = 0;
    int64_t kmax = p.max_steps;  // step budget of this run (SLICED: of the current slice)

    // SLICED: another SM wrote these rows in the previous slice; read them from L2, never from a stale L1 line
    auto ld = [](const auto* q) {
        if constexpr (SLICED) return __ldcg(q);
        else return *q;
    };
    auto load_system = [&]() {  // sys -> registers; sets active / writeback
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const int gid = l * B + b;
            // dummy slot (padded shapes only): massless, at rest, far from everything and from each other
            X[b][0] = 1.0e8 * (double)(gid + 1);
            X[b][1] = X[b][2] = 0.0;
            V[b][0] = V[b][1] = V[b][2] = 0.0;
            m[b] = 0.0;
            if (!PADDED || gid < N) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    X[b][c] = ld(&e.pos[(int64_t)(gid * 3 + c) * e.n_pad + sys]);
                    V[b][c] = ld(&e.vel[(int64_t)(gid * 3 + c) * e.n_pad + sys]);
                }
                m[b] = e.mass[(int64_t)gid * e.n_pad + sys];
            }
        }
        {
            const double t = ld(&e.time[sys]);
            ts = fwd ? t : -t;
        }
        st = ld(&e.status[sys]);
        k = 0;
        active = st < ENS_STOP_CLOSE;  // STOP_* are sticky; DONE_* run again
        writeback = active;
    };
    auto store_system = [&]() {  // registers -> sys (only systems that were advanced)
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
                e.nsteps[sys] = ld(&e.nsteps[sys]) + k;
            }
        }
        writeback = false;
    };

    bool exhausted = !(sl < S);  // ADAPT: this lane group will pull no more systems
    if constexpr (!ADAPT && !SLICED) {
#pragma unroll
        for (int b = 0; b < B; ++b) {
            X[b][0] = 1.0e8 * (double)(l * B + b + 1);
            X[b][1] = X[b][2] = 0.0;
            V[b][0] = V[b][1] = V[b][2] = 0.0;
            m[b] = 0.0;
        }
        if ((sl < S) && (sys < e.n_sys)) load_system();
    }
    // ADAPT only; called with the whole warp converged, at step boundaries: groups without a running system store
    // the one they finished and pull the next index
    auto refill = [&]() -> bool {
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
        return __ballot_sync(0xffffffffu, !exhausted) != 0;  // somebody may still be running or pulling
    };

    // Eq. 3 / Eq. 4 with the step-size powers folded in (algebraically the oracle's formulas):
    //   x_p = x + h v + h^2/2 a0 + h^3/6 j0          v_p = v + h a0 + h^2/2 j0
    //   C_x = x + h v + 7/20 h^2 a0 + 1/20 h^3 j0    C_v = v + h/2 a0 + 1/12 h^2 j0
    //   x_c = C_x + 3/20 h^2 a1 - 1/30 h^3 j1        v_c = C_v + h/2 a1 - 1/12 h^2 j1
    // The ten coefficients come precomputed in StepArgs (constant bank operands of the DFMAs: no registers).
    double h = p.dt;  // the step taken; ADAPT: recomputed from (a0, j0) at the start of every step

    double Cx[B][3], Cv[B][3];
    double a[B][3], j[B][3];
    unsigned r2min;  // high word of the smallest squared pair separation seen by the last tracking evaluation

    // Phase 0 of a step, in three parts.  X, V hold the accepted state.
    // quick_test: monitors act on post-step states only (Alg. 1: advance, then execute(M)).  Nearly every step of nearly
    // every system has nothing to report, so the step loop carries ONE test, one vote and one warp-uniform, almost never
    // taken branch: a lane is `quiet` when every pair it saw is farther apart than r_close (high word of r^2 strictly
    // above the threshold's: the exact 64-bit decision cannot differ) and every coordinate of its bodies is below
    // r_eject / sqrt(3) (high words of the coordinates, integer ALU; StepArgs::ce_hi: then |x|^2 < r_eject^2 and finite;
    // non-finite values sort above every finite one), and `go` when it is quiet, has time left and steps left.  Returns
    // the lanes of amask that are not `go`; only when there is one does the warp run exact_stop.
    auto quick_test = [&](unsigned amask) -> unsigned {
        unsigned cmax = 0u;  // largest high word of the |coordinates| of the bodies of this lane
#pragma unroll
        for (int b = 0; b < B; ++b)
#pragma unroll
            for (int c = 0; c < 3; ++c)
                if (!PADDED || (l * B + b < N)) cmax = max(cmax, (unsigned)__double2hiint(X[b][c]) & 0x7fffffffu);
        const bool go = (r2min > (unsigned)(p.rc2_bits >> 32)) && (cmax < p.ce_hi) && (ts < p.te) && (k < kmax);
        return __ballot_sync(amask, !go);
    };
    // exact_stop: the exact monitor / stop logic (also resolves high-word ties); updates `active` and `st`.  Every lane
    // of amask takes part in the flag reduction (with refilled systems k differs between the systems of a warp).
    auto exact_stop = [&](unsigned amask) {
        const int f = monitor_flags<N, L, B>(X, r2min, p, l, base, amask);
        if (k > 0 && f) {
            st = (f & 4) ? ENS_STOP_NONFINITE : (f & 1) ? ENS_STOP_CLOSE : ENS_STOP_EJECT;
            active = false;
        }
        if (active) {
            if (!(ts < p.te)) {
                st = ENS_DONE_TIME;
                active = false;
            } else if (k >= kmax) {
                st = ENS_DONE_STEPS;
                active = false;
            }
        }
    };
    // predict: the step is now certain to be taken, so its bookkeeping (time, step count) is done here, a whole step
    // ahead of the quick test that reads it.  am2 = the lanes that take the step.
    auto predict = [&](unsigned am2) {
        double p_a = p.p_a, p_j = p.p_j, cx_a = p.cx_a, cx_j = p.cx_j, cv_a = p.cv_a, cv_j = p.cv_j;
        if constexpr (ADAPT) {
            h = adaptive_dt<N, L, B>(a, j, p.dt, l, base, am2);
            const double h2 = h * h, h3 = h2 * h;
            p_a = 0.5 * h2;
            p_j = (1.0 / 6.0) * h3;
            cx_a = 0.35 * h2;
            cx_j = 0.05 * h3;
            cv_a = 0.5 * h;
            cv_j = (1.0 / 12.0) * h2;
        }
        if constexpr (UNROLL) {  // (the 3-phase loop does it in its last phase: fewer values live across the evaluations)
            ts += fabs(h);       // h carries the sign of the direction
            ++k;
        }
#pragma unroll
        for (int b = 0; b < B; ++b)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double tx = fma(h, V[b][c], X[b][c]);
                Cx[b][c] = fma(cx_j, j[b][c], fma(cx_a, a[b][c], tx));
                Cv[b][c] = fma(cv_j, j[b][c], fma(cv_a, a[b][c], V[b][c]));
                X[b][c] = fma(p_j, j[b][c], fma(p_a, a[b][c], tx));
                V[b][c] = fma(p_a, j[b][c], fma(h, a[b][c], V[b][c]));
            }
    };
    auto accept_and_predict = [&](unsigned amask) {
        if (__builtin_expect(quick_test(amask) != 0u, 0)) exact_stop(amask);
        // lanes that just stopped take no part in the shuffles of predict: re-vote (every lane of amask is here)
        unsigned am2 = amask;
        if constexpr (ADAPT && L > 1) am2 = __ballot_sync(amask, active);
        if (active) predict(am2);
    };
    auto correct = [&]() {
        double kx_a = p.kx_a, kx_j = p.kx_j, kv_a = p.kv_a, kv_j = p.kv_j;
        if constexpr (ADAPT) {  // rebuilt from h each time: one live register pair instead of four
            const double h2 = h * h;
            kx_a = 0.15 * h2;
            kx_j = (-1.0 / 30.0) * (h2 * h);
            kv_a = 0.5 * h;
            kv_j = (-1.0 / 12.0) * h2;
        }
#pragma unroll
        for (int b = 0; b < B; ++b)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                X[b][c] = fma(kx_j, j[b][c], fma(kx_a, a[b][c], Cx[b][c]));
                V[b][c] = fma(kv_j, j[b][c], fma(kv_a, a[b][c], Cv[b][c]));
            }
    };

    // the two corrector iterations of the straight-line kernels: two inlined copies (UNROLL = 1) or one copy in a loop
    // (UNROLL = 2: a third less code to fetch per step; faster where the straight-line step outgrows the instruction
    // cache, n_body = 6: 35 KB)
    auto corrector_iterations = [&](unsigned am) {
        if constexpr (UNROLL == 2) {
#pragma unroll 1
            for (int it = 0; it < 2; ++it) {
                eval_acc_jerk<N, L, B, false>(X, V, m, a, j, r2min, l, base, am, W);
                correct();
            }
        } else {
            eval_acc_jerk<N, L, B, false>(X, V, m, a, j, r2min, l, base, am, W);
            correct();
            eval_acc_jerk<N, L, B, false>(X, V, m, a, j, r2min, l, base, am, W);
            correct();
        }
    };
    bool fresh = true;  // CARRY: a, j do not yet belong to the current state (warp-uniform: start of the launch)
    auto run = [&]() {
    if constexpr (UNROLL && !ADAPT) {
        // Straight-line step, fixed step size: the systems of the warp that run enter the loop together (mask am) and
        // stay in it until the exact stop logic retires them; it runs only when the quick test fails for some lane, so a
        // step costs one vote, one almost never taken branch and the loop's jump.
        const unsigned amask0 = __ballot_sync(0xffffffffu, active);
        if (active) {
            unsigned am = amask0;
            if constexpr (CARRY) {  // the one evaluation at the state itself (start of the launch), outside the loop
                eval_acc_jerk<N, L, B>(X, V, m, a, j, r2min, l, base, am, W);
                fresh = false;
            }
            while (true) {
                if constexpr (!CARRY) eval_acc_jerk<N, L, B>(X, V, m, a, j, r2min, l, base, am, W);
                if (__builtin_expect(quick_test(am) != 0u, 0)) {
                    exact_stop(am);
                    am = __ballot_sync(am, active);  // the lanes that go on
                    if (!active) break;
                }
                predict(am);
                corrector_iterations(am);
                // CARRY: (a, j) of the last corrector evaluation open the next step; its monitor needs the separations
                // of the post-step state
                if constexpr (CARRY) r2min = p.rc2_bits ? (unsigned)(pair_r2min<N, L, B>(X, l, base, am) >> 32) : ~0u;
            }
        }
    } else if constexpr (UNROLL) {
        // Straight-line step, adaptive step size (persistent grid).  The groups that hold a system run the same inner
        // loop as above; when the exact stop logic retires a system the whole warp leaves it (a warp-uniform break), so
        // that the idle group pulls its next system at this step boundary.  The groups that go on re-enter and repeat
        // the evaluation they had just done (same state, same result, bit for bit): one evaluation per retirement
        // and warp, about 0.5 % of the work of a launch.
        while (refill()) {
            const unsigned amask = __ballot_sync(0xffffffffu, active);
            if (amask == 0) continue;
            if (active) {
                while (true) {
                    eval_acc_jerk<N, L, B>(X, V, m, a, j, r2min, l, base, amask, W);
                    if (__builtin_expect(quick_test(amask) != 0u, 0)) {
                        exact_stop(amask);
                        if (__ballot_sync(amask, active) != amask) break;  // some group retired its system
                    }
                    predict(amask);
                    corrector_iterations(amask);
                }
            }
        }
    } else {
        int phase = 0;  // warp-uniform: 0 = accept + predict, 1 and 2 = corrector iterations
        while (true) {
            if constexpr (ADAPT) {
                if (phase == 0 && !refill()) break;
            }
            const unsigned amask = __ballot_sync(0xffffffffu, active);
            if (amask == 0) {
                if constexpr (ADAPT) {
                    phase = 0;
                    continue;
                }
                break;
            }
            if (active) {
                if (!CARRY || fresh || phase != 0)
                    eval_acc_jerk<N, L, B>(X, V, m, a, j, r2min, l, base, amask, W);
                else
                    r2min = p.rc2_bits ? (unsigned)(pair_r2min<N, L, B>(X, l, base, amask) >> 32) : ~0u;
                if (phase == 0) {
                    accept_and_predict(amask);
                } else {
                    correct();
                    if (phase == 2) {
                        ts += fabs(h);
                        ++k;
                    }
                }
            }
            phase = phase == 2 ? 0 : phase + 1;
            fresh = false;
        }
    }
    };
    if constexpr (SLICED) {
        const unsigned long long G = (unsigned long long)p.n_groups, n_tasks = G * (unsigned long long)p.n_slices;
        while (true) {
            unsigned long long task = 0;
            if (lane == 0) task = atomicAdd(p.counter, 1ull);
            task = __shfl_sync(0xffffffffu, task, 0);
            if (task >= n_tasks) break;
            const int64_t s = (int64_t)(task / G), g = (int64_t)(task - (unsigned long long)s * G);
            if (s > 0) {  // slice s - 1 of this group is held by a running warp (tasks are handed out in order)
                if (lane == 0) {
                    int seen;
                    while (true) {
                        asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(seen) : "l"(p.slice_done + g) : "memory");
                        if (seen >= (int)s) break;
                        __nanosleep(200);
                    }
                }
                __syncwarp();
            }
            sys = g * S + sl;
#pragma unroll
            for (int b = 0; b < B; ++b) {
                X[b][0] = 1.0e8 * (double)(l * B + b + 1);
                X[b][1] = X[b][2] = 0.0;
                V[b][0] = V[b][1] = V[b][2] = 0.0;
                m[b] = 0.0;
            }
            active = writeback = false;
            if ((sl < S) && (sys < e.n_sys)) {
                load_system();
                // a system that ran out of time in an earlier slice of this call is still out of time
                if (s > 0 && st == ENS_DONE_TIME) active = writeback = false;
            }
            const int64_t left = p.max_steps - s * p.slice_steps;
            kmax = (left < p.slice_steps || s == p.n_slices - 1) ? left : p.slice_steps;  // the last slice is open-ended
            run();
            store_system();
            __threadfence();
            __syncwarp();
            if (lane == 0) asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p.slice_done + g), "r"((int)s + 1) : "memory");
        }
    } else {
        run();
        store_system();
    }
}

}  // namespace ensd
