// acc_pairs.cuh — acceleration-only pair evaluation over the bodies a group of L lanes holds (Eq. 1, R1), each
// unordered pair once: in-lane pairs in registers, cross-lane pairs by the lane ring of the Hermite kernel
// (visitors through shared memory, returned halves by shuffle).  Used by the MVS kernel (planet-planet accelerations; the star's pull is in the Kepler drift) and by
// the Runge-Kutta kernel (all bodies).
#pragma once
#include "ens_device.cuh"

namespace ensd {

// One unordered planet pair (i, k), acceleration only: a_i += m_k dx / r^3, a_k -= m_i dx / r^3  (Eq. 1, R1).
// FIRST_K = true: a_k is assigned, not accumulated (the visitor's sum starts with this pair).
template <bool FIRST_K = false>
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
        if constexpr (FIRST_K) ak[c] = wk * dx[c];
        else ak[c] = fma(wk, dx[c], ak[c]);
    }
    return r2;
}

// the tracked minimum's high word, and the exact minimum (recomputed from the positions when only the high word was kept)
__device__ __forceinline__ unsigned r2_high_word(u64 v) { return (unsigned)(v >> 32); }
__device__ __forceinline__ unsigned r2_high_word(unsigned v) { return v; }
template <int N, int L, int B>
__device__ __forceinline__ u64 r2_exact(u64 tracked, const double (&)[B][3], int, int, unsigned) {
    return tracked;
}
template <int N, int L, int B>
__device__ __forceinline__ u64 r2_exact(unsigned, const double (&x)[B][3], int l, int base, unsigned mask) {
    return pair_r2min<N, L, B>(x, l, base, mask);
}

// Shared memory of the cross-lane schedule (L > 1 only), per warp, in 16-byte words, word-major (word w of lane n at
// [w * 32 + n]):  B * 2 words per lane: (x0, x1) (x2, m) of each of the lane's bodies.
template <int L, int B>
__host__ __device__ constexpr int acc_ring_smem_words() {
    return L > 1 ? B * 2 * 32 : 0;
}

// Planet-planet accelerations of the B planets this lane owns (the star's pull is in the Kepler drift).
// In-lane pairs in (b ascending, c ascending) order give every planet its contributions in ascending k, the
// oracle's order, when L = 1.  Cross-lane pairs (L > 1) as in hermite_kernel.cuh: every lane publishes its bodies in
// shared memory (W = this warp's acc_ring_smem_words) and reads the visiting body right before the B pairs that use it;
// the visitor's halves go back by shuffle and are added one visit behind, so that no instruction waits on a shuffle
// that was just issued.
template <int P, int L, int B, class R2>
__device__ __forceinline__ void eval_acc_planets(const double (&Q)[B][3], const double (&m)[B], double (&A)[B][3],
                                                 R2& r2min, int l, int base, unsigned amask, double2* W) {
    constexpr bool PADDED = (L * B != P);
#pragma unroll
    for (int b = 0; b < B; ++b) A[b][0] = A[b][1] = A[b][2] = 0.0;
    // r2min: the smallest squared separation this lane saw, tracked on the integer ALU either as the HIGH WORD of its bit
    // pattern (R2 = unsigned: one integer min per pair; pair_r2min gives the exact value when the stop logic needs it) or
    // as the full pattern (R2 = u64: a 64-bit compare and select per pair).  The caller chooses: the high word is faster
    // for the one-system-per-thread shapes, the many-lane Cash-Karp shapes are faster with the full pattern (measured).
    r2min = (R2)~(R2)0;
    auto track = [&](double r2, bool valid) {
        if constexpr (sizeof(R2) == 8) min_bits(r2min, r2, valid);
        else min_hi(r2min, r2, valid);
    };
    if constexpr (L > 1) {
        const int wl = threadIdx.x & 31;
        __syncwarp(amask);  // every lane has finished reading the previous publication
#pragma unroll
        for (int c = 0; c < B; ++c) {
            W[(c * 2 + 0) * 32 + wl] = make_double2(Q[c][0], Q[c][1]);
            W[(c * 2 + 1) * 32 + wl] = make_double2(Q[c][2], m[c]);
        }
        __syncwarp(amask);
    }
#pragma unroll
    for (int b = 0; b < B; ++b)
#pragma unroll
        for (int c = b + 1; c < B; ++c) {
            const double r2 = pair_acc(Q[b], m[b], A[b], Q[c], m[c], A[c]);
            track(r2, !PADDED || (l * B + c < P));
        }
    if constexpr (L > 1) {
        constexpr int H = (L - 1) / 2;
        double ra[3];  // the other half of the pairs of ONE of my bodies, computed by lane l - s; in flight
#pragma unroll
        for (int s = 1; s <= H; ++s) {
            int ls = l + s;
            if (ls >= L) ls -= L;
            int lr = l - s;
            if (lr < 0) lr += L;
            const int src = base + ls, ret = base + lr;
#pragma unroll
            for (int c = 0; c < B; ++c) {
                const int vis = (s - 1) * B + c;
                const double2 w0 = W[(c * 2 + 0) * 32 + src], w1 = W[(c * 2 + 1) * 32 + src];
                const double xv[3] = {w0.x, w0.y, w1.x};
                const double mv = w1.y;
                double av[3];  // the visitor's half of these B pairs: started by the first pair
                const bool vvalid = !PADDED || (ls * B + c < P);
#pragma unroll
                for (int b = 0; b < B; ++b) {
                    const double r2 = b == 0 ? pair_acc<true>(Q[b], m[b], A[b], xv, mv, av) : pair_acc(Q[b], m[b], A[b], xv, mv, av);
                    track(r2, vvalid && (!PADDED || (l * B + b < P)));
                }
                if (vis >= 1) {  // sent one visit ago
#pragma unroll
                    for (int q = 0; q < 3; ++q) A[(vis - 1) % B][q] += ra[q];
                }
#pragma unroll
                for (int q = 0; q < 3; ++q) ra[q] = __shfl_sync(amask, av[q], ret);
            }
        }
#pragma unroll
        for (int q = 0; q < 3; ++q) A[B - 1][q] += ra[q];
    }
}

}  // namespace ensd
