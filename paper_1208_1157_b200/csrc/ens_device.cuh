// ens_device.cuh — device helpers shared by the Hermite and MVS kernels (CUDA path only; nothing here is used by oracle/).
#pragma once
#include "ens_internal.cuh"

namespace ensd {

typedef unsigned long long u64;

__device__ __forceinline__ u64 dbits(double x) { return (u64)__double_as_longlong(x); }

// FP64 reciprocal square root (P:L276 used the Fermi hardware rsqrt; R14): MUFU.RSQ seed of the value rounded
// to FP32 (relative error <= 2^-22) and one cubic Newton-Halley step in FP64,
//   e = 1 - r2 y0^2,  y = y0 + y0 e (1/2 + 3/8 e),   remaining error ~ (5/16) e^3 < 2^-66 plus rounding: <= 1 ulp
// (tests/test_gpu_device_functions.py measures it).  Valid for r2 inside the FP32 normal range, 1.2e-38 < r2 <
// 3.4e38, i.e. separations between 1e-19 and 1e19 length units.
__device__ __forceinline__ double rsqrt_f64(double r2) {
    float s;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(s) : "f"(__double2float_rn(r2)));
    const double y0 = (double)s;
    const double t = r2 * y0;
    const double e = fma(-t, y0, 1.0);
    const double p = fma(0.375, e, 0.5);
    const double q = y0 * e;
    return fma(q, p, y0);
}

// FP64 reciprocal without the IEEE divide sequence: MUFU.RCP seed of the value rounded to FP32 (relative error
// <= 2^-22), then y = y0 + y0 e (1 + e), e = 1 - x y0: remaining error e^3 < 2^-66 plus rounding (<= 1 ulp).
// REFINE = false stops at y0 + y0 e (relative error 2^-44): enough for a Newton step, which is self-correcting.
// Valid for |x| inside the FP32 normal range.
template <bool REFINE>
__device__ __forceinline__ double rcp_f64(double x) {
    float s;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(s) : "f"(__double2float_rn(x)));
    const double y0 = (double)s;
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

}  // namespace ensd
