// ens_device.cuh — device helpers shared by the Hermite and MVS kernels (CUDA path only; nothing here is used by oracle/).
#pragma once
#include "ens_internal.cuh"

namespace ensd {

typedef unsigned long long u64;

__device__ __forceinline__ u64 dbits(double x) { return (u64)__double_as_longlong(x); }

// FP64 reciprocal square root (P:L276 used the Fermi hardware rsqrt; R14): MUFU.RSQ64H seed (the approximation unit
// reads the high word of the double: no F2F round trip, full FP64 exponent range, relative error ~2^-20) and one
// cubic Newton-Halley step in FP64,
//   e = 1 - r2 y0^2,  y = y0 + y0 e (1/2 + 3/8 e),   remaining error ~ (5/16) e^3 < 2^-61 plus rounding: <= 1 ulp
// (tests/test_gpu_hermite.py::test_rsqrt_within_one_ulp measures it).  Valid for normal, finite r2 > 0.
// (An FP32 seed - MUFU.RSQ of the value rounded to float, two extra F2F per call, r2 restricted to the FP32 range - was
// 2-6 % slower in every kernel: DESIGN.md section 8.)
__device__ __forceinline__ double rsqrt_f64(double r2) {
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(r2));
    const double t = r2 * y0;
    const double e = fma(-t, y0, 1.0);
    const double p = fma(0.375, e, 0.5);
    const double q = y0 * e;
    return fma(q, p, y0);
}

// FP64 reciprocal without the IEEE divide sequence: MUFU.RCP64H seed (relative error ~2^-20), then
// y = y0 + y0 e (1 + e), e = 1 - x y0: remaining error e^3 < 2^-60 plus rounding (<= 1 ulp).
// REFINE = false stops at y0 + y0 e (relative error ~2^-40): enough for a Newton step, which is self-correcting.
// Valid for normal, finite x != 0.
template <bool REFINE>
__device__ __forceinline__ double rcp_f64(double x) {
    double y0;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(x));
    const double e = fma(-x, y0, 1.0);
    const double q = y0 * e;
    if constexpr (REFINE) return fma(q, 1.0 + e, y0);
    return y0 + q;
}

__device__ __forceinline__ void min_bits(u64& acc, double r2, bool valid = true) {
    // r2 >= 0 or NaN: unsigned order of the bit patterns is the numeric order and NaN sorts above +inf, so this
    // minimum runs on the integer ALU, not the FP64 pipe.
    const u64 b = valid ? dbits(r2) : ~0ull;
    acc = b < acc ? b : acc;
}

// The same minimum on the high words only (exponent and top 20 mantissa bits): one integer min per value.  Exact
// whenever the compared high words differ; the caller resolves ties (hermite_kernel.cuh: monitor_flags).
__device__ __forceinline__ void min_hi(unsigned& acc, double r2, bool valid = true) {
    const unsigned h = valid ? (unsigned)__double2hiint(r2) : ~0u;
    acc = min(acc, h);
}


// Smallest squared pair separation of the N bodies a group of L lanes holds (bit pattern), positions only, in the
// arithmetic of the pair evaluations (dx = x_k - x_i; r^2 = fma(dz, dz, fma(dy, dy, dx dx))): the exact value behind
// the high words the step loops track.  Used by the exact stop logic of every kernel and by the close-approach monitor
// of the 2-evaluation Hermite variant.  Same lane ring as the evaluations, by shuffle; no return traffic (each lane
// keeps the minimum over the pairs it sees; the caller reduces the flag over the lanes).
template <int N, int L, int B>
__device__ __forceinline__ u64 pair_r2min(const double (&x)[B][3], int l, int base, unsigned amask) {
    constexpr bool PADDED = (L * B != N);
    u64 r2min = ~0ull;
    auto d2 = [](const double (&p)[3], const double (&q)[3]) {
        const double dx = q[0] - p[0], dy = q[1] - p[1], dz = q[2] - p[2];
        return fma(dz, dz, fma(dy, dy, dx * dx));
    };
#pragma unroll
    for (int b = 0; b < B; ++b)
#pragma unroll
        for (int c = b + 1; c < B; ++c) min_bits(r2min, d2(x[b], x[c]), !PADDED || (l * B + c < N));
    if constexpr (L > 1) {
#pragma unroll
        for (int s = 1; s <= (L - 1) / 2; ++s) {
            int ls = l + s;
            if (ls >= L) ls -= L;
#pragma unroll
            for (int c = 0; c < B; ++c) {
                double xv[3];
#pragma unroll
                for (int q = 0; q < 3; ++q) xv[q] = __shfl_sync(amask, x[c][q], base + ls);
                const bool vvalid = !PADDED || (ls * B + c < N);
#pragma unroll
                for (int b = 0; b < B; ++b) min_bits(r2min, d2(x[b], xv), vvalid && (!PADDED || (l * B + b < N)));
            }
        }
    }
    return r2min;
}

}  // namespace ensd
