// adaptive_order.cu — hand-out order of the systems for the adaptive-step Hermite kernel.
//
// The adaptive kernel runs a persistent grid whose lane groups pull system indices from a counter.  A launch
// integrates only one or two systems per lane group, so the order of hand-out decides the end-of-launch tail:
// longest first (the LPT rule) lets the short systems fill the gaps.  The expected work of a system is the number of
// steps it will take, estimated as |t_end - t| / dt_0 with dt_0 the step Eq. 5 gives for its initial
// state — i.e. |t_end - t| sqrt(sum_i |j_i|^2 / |a_i|^2) / tau, the tau dropped.  The estimate only orders the work:
// results do not depend on it (systems are independent and each is integrated by the same code whatever its slot).
// The sort is a library primitive (cub::DeviceRadixSort); the keys come from the kernel below.
#include <cub/device/device_radix_sort.cuh>

#include "ens_internal.cuh"

namespace ensd {

namespace {

// one thread per system, plain double loop over the pairs (n_body is a run-time value here: this runs once per launch)
__global__ void __launch_bounds__(128) order_key_kernel(View e, double t_end, float* __restrict__ key,
                                                        int32_t* __restrict__ idx) {
    const int64_t sys = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (sys >= e.n_sys) return;
    const int n = e.n_body;
    double x[16][3], v[16][3], m[16];
    for (int i = 0; i < n; ++i) {
        for (int c = 0; c < 3; ++c) {
            x[i][c] = e.pos[(int64_t)(i * 3 + c) * e.n_pad + sys];
            v[i][c] = e.vel[(int64_t)(i * 3 + c) * e.n_pad + sys];
        }
        m[i] = e.mass[(int64_t)i * e.n_pad + sys];
    }
    double sum = 0.0;
    for (int i = 0; i < n; ++i) {
        double a[3] = {0.0, 0.0, 0.0}, j[3] = {0.0, 0.0, 0.0};
        for (int k = 0; k < n; ++k) {
            if (k == i) continue;
            const double dx = x[k][0] - x[i][0], dy = x[k][1] - x[i][1], dz = x[k][2] - x[i][2];
            const double du = v[k][0] - v[i][0], dv = v[k][1] - v[i][1], dw = v[k][2] - v[i][2];
            const double r2 = dx * dx + dy * dy + dz * dz, rv = dx * du + dy * dv + dz * dw;
            const double y = rsqrt(r2), w = m[k] * y * y * y, s = -3.0 * rv * y * y;
            a[0] += w * dx;
            a[1] += w * dy;
            a[2] += w * dz;
            j[0] += w * (du + s * dx);
            j[1] += w * (dv + s * dy);
            j[2] += w * (dw + s * dz);
        }
        const double a2 = a[0] * a[0] + a[1] * a[1] + a[2] * a[2], j2 = j[0] * j[0] + j[1] * j[1] + j[2] * j[2];
        if (a2 > 0.0) sum += j2 / a2;
    }
    double span = fabs(t_end - e.time[sys]);
    if (!(span < 1e300)) span = 1.0;  // pure step-count control: every system takes the same number of steps
    const int st = e.status[sys];
    float kf = (float)(span * sqrt(sum));
    if (!(kf >= 0.0f) || st >= ENS_STOP_CLOSE) kf = 0.0f;  // NaN, or a system that will not run: last
    key[sys] = kf;
    idx[sys] = (int32_t)sys;
}

}  // namespace

// All buffers of the hand-out order for n systems (called by ens_create, so that ens_integrate never allocates).  On any
// failure everything is released again: `ob` is either complete or empty.
cudaError_t adaptive_order_alloc(int64_t n_sys, OrderBuffers& ob) {
    const int n = (int)n_sys;
    cudaError_t err = cudaSuccess;
    if ((err = cudaMalloc(&ob.key_in, sizeof(float) * n)) == cudaSuccess &&
        (err = cudaMalloc(&ob.key_out, sizeof(float) * n)) == cudaSuccess &&
        (err = cudaMalloc(&ob.idx_in, sizeof(int32_t) * n)) == cudaSuccess &&
        (err = cudaMalloc(&ob.idx_out, sizeof(int32_t) * n)) == cudaSuccess &&
        (err = cub::DeviceRadixSort::SortPairsDescending(nullptr, ob.tmp_bytes, ob.key_in, ob.key_out, ob.idx_in,
                                                         ob.idx_out, n, 0, 32, (cudaStream_t)0)) == cudaSuccess)
        err = cudaMalloc(&ob.tmp, ob.tmp_bytes ? ob.tmp_bytes : 1);
    if (err != cudaSuccess) adaptive_order_free(ob);
    return err;
}

cudaError_t adaptive_order(const View& v, double t_end, OrderBuffers& ob, cudaStream_t s) {
    if (!ob.key_in || !ob.key_out || !ob.idx_in || !ob.idx_out || !ob.tmp) return cudaErrorInvalidValue;
    cudaError_t err = cudaSuccess;
    const int n = (int)v.n_sys;
    order_key_kernel<<<(unsigned)((v.n_sys + 127) / 128), 128, 0, s>>>(v, t_end, ob.key_in, ob.idx_in);
    if ((err = cudaGetLastError()) != cudaSuccess) return err;
    return cub::DeviceRadixSort::SortPairsDescending(ob.tmp, ob.tmp_bytes, ob.key_in, ob.key_out, ob.idx_in, ob.idx_out,
                                                     n, 0, 32, s);
}

void adaptive_order_free(OrderBuffers& ob) {
    cudaFree(ob.key_in);
    cudaFree(ob.key_out);
    cudaFree(ob.idx_in);
    cudaFree(ob.idx_out);
    cudaFree(ob.tmp);
    ob = OrderBuffers();
}

}  // namespace ensd
