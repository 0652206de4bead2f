// acc_pairs.cuh — acceleration-only pair evaluation over the bodies a group of L lanes holds (Eq. 1, R1), each
// unordered pair once: in-lane pairs in registers, cross-lane pairs by the ring of shuffles of the Hermite
// kernel.  Used by the MVS kernel (planet-planet accelerations; the star's pull is in the Kepler drift) and by
// the Runge-Kutta kernel (all bodies).
#pragma once
#include "ens_device.cuh"

namespace ensd {

// One unordered planet pair (i, k), acceleration only: a_i += m_k dx / r^3, a_k -= m_i dx / r^3  (Eq. 1, R1).
__device__ __forceinline__ double pair_acc(const double (&xi)[3], double mi, double (&ai)[3], const double (&xk)[3],
                                           double mk, double (&ak)[3]) {
    double dx[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) dx[c] = xk[c] - xi[c];
    const double r2 = fma(dx[2], dx[2], fma(dx[1], dx[1], dx[0] * dx[0]));
    const double y = rsqrt_f64(r2);
    const double y3 = y * y * y;
    const double wi = mk * y3;
    const double wk = -mi * y3;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        ai[c] = fma(wi, dx[c], ai[c]);
        ak[c] = fma(wk, dx[c], ak[c]);
    }
    return r2;
}

// Planet-planet accelerations of the B planets this lane owns (the star's pull is in the Kepler drift).
// In-lane pairs in (b ascending, c ascending) order give every planet its contributions in ascending k, the
// oracle's order, when L = 1.
template <int P, int L, int B>
__device__ __forceinline__ void eval_acc_planets(const double (&Q)[B][3], const double (&m)[B], double (&A)[B][3],
                                                 u64& r2min, int l, int base, unsigned amask) {
    constexpr bool PADDED = (L * B != P);
#pragma unroll
    for (int b = 0; b < B; ++b) A[b][0] = A[b][1] = A[b][2] = 0.0;
    r2min = ~0ull;
#pragma unroll
    for (int b = 0; b < B; ++b)
#pragma unroll
        for (int c = b + 1; c < B; ++c) {
            const double r2 = pair_acc(Q[b], m[b], A[b], Q[c], m[c], A[c]);
            min_bits(r2min, r2, !PADDED || (l * B + c < P));
        }
    if constexpr (L > 1) {
#pragma unroll
        for (int s = 1; s <= (L - 1) / 2; ++s) {
            int ls = l + s;
            if (ls >= L) ls -= L;
            int lr = l - s;
            if (lr < 0) lr += L;
            const int src = base + ls, ret = base + lr;
#pragma unroll
            for (int c = 0; c < B; ++c) {
                double xv[3], av[3] = {0.0, 0.0, 0.0};
#pragma unroll
                for (int q = 0; q < 3; ++q) xv[q] = __shfl_sync(amask, Q[c][q], src);
                const double mv = __shfl_sync(amask, m[c], src);
                const bool vvalid = !PADDED || (ls * B + c < P);
#pragma unroll
                for (int b = 0; b < B; ++b) {
                    const double r2 = pair_acc(Q[b], m[b], A[b], xv, mv, av);
                    min_bits(r2min, r2, vvalid && (!PADDED || (l * B + b < P)));
                }
#pragma unroll
                for (int q = 0; q < 3; ++q) A[c][q] += __shfl_sync(amask, av[q], ret);
            }
        }
    }
}

}  // namespace ensd
