// hermite.cu — instantiations of the fused Hermite step-loop kernel and the n_body -> (L, B) dispatch.
#include "hermite_kernel.cuh"

namespace ensd {

namespace {

// n_body -> lanes per system L (odd), bodies per lane B, L * B >= n_body.  Exact fits for 2-6, 9, 10, 12, 15;
// the others run in the next larger shape with massless dummy slots.
template <int N> struct ShapeOf;
#define ENS_SHAPE(N_, L_, B_, UNROLL_, THREADS_, MINB_) ENS_SHAPE_T(N_, L_, B_, UNROLL_, THREADS_, MINB_, 128)
#define ENS_SHAPE_T(N_, L_, B_, UNROLL_, THREADS_, MINB_, MAXT_)                        \
    template <> struct ShapeOf<N_> {                                                    \
        static constexpr int L = L_, B = B_, THREADS = THREADS_, MINB = MINB_, MAXT = MAXT_; \
        static constexpr bool UNROLL = UNROLL_;                                         \
    };
// Tuning knobs of the headline shape (n_body = 3), overridable at compile time for the sweeps recorded in DESIGN.md §8.
#ifndef ENS_H3_UNROLL
#define ENS_H3_UNROLL true
#endif
#ifndef ENS_H3_THREADS
#define ENS_H3_THREADS 64
#endif
#ifndef ENS_H3_MAXT
#define ENS_H3_MAXT 64  // __launch_bounds__ threads: with MINB it sets the register cap 65536 / (MAXT * MINB)
#endif
#ifndef ENS_H3_MINB
#define ENS_H3_MINB 7  // register cap 128 (125 used, no spills), 8 blocks of 2 warps per SM (sweeps: DESIGN.md §8)
#endif
//        N  L  B  unroll threads minBlocks
ENS_SHAPE(2, 1, 2, true, 64, 1)
ENS_SHAPE_T(3, 1, 3, ENS_H3_UNROLL, ENS_H3_THREADS, ENS_H3_MINB, ENS_H3_MAXT)
ENS_SHAPE(4, 1, 4, true, 64, 1)
ENS_SHAPE(5, 1, 5, true, 64, 1)
// n_body = 6 (config 2): one system per thread, all 15 pairs in one lane, no shuffles: 0.62 of FP64 issue peak against
// 0.54 for the best 3-lane shape; 32-thread blocks spread the 1024 warps of config 2 evenly over the SMs.
#ifndef ENS_H6_L
#define ENS_H6_L 1
#define ENS_H6_B 6
#endif
#ifndef ENS_H6_THREADS
#define ENS_H6_THREADS 32
#define ENS_H6_MAXT 32
#define ENS_H6_MINB 1
#endif
#ifndef ENS_H6_UNROLL
#define ENS_H6_UNROLL true  // straight-line step (three copies of the 15-pair evaluation): 0.668 against 0.653 for the 3-phase loop
#endif
ENS_SHAPE_T(6, ENS_H6_L, ENS_H6_B, ENS_H6_UNROLL, ENS_H6_THREADS, ENS_H6_MINB, ENS_H6_MAXT)
ENS_SHAPE(7, 3, 3, false, 64, 1)
ENS_SHAPE(8, 3, 3, false, 64, 1)
ENS_SHAPE(9, 3, 3, false, 64, 1)
ENS_SHAPE(10, 5, 2, false, 64, 1)
ENS_SHAPE(11, 3, 4, false, 64, 1)
ENS_SHAPE(12, 3, 4, false, 64, 1)
ENS_SHAPE(13, 5, 3, false, 64, 1)
ENS_SHAPE(14, 5, 3, false, 64, 1)
#ifndef ENS_H15_L
#define ENS_H15_L 5
#define ENS_H15_B 3
#endif
#ifndef ENS_H15_THREADS
#define ENS_H15_THREADS 64
#define ENS_H15_MAXT 128
#define ENS_H15_MINB 1
#endif
#ifndef ENS_H15_UNROLL
#define ENS_H15_UNROLL false
#endif
ENS_SHAPE_T(15, ENS_H15_L, ENS_H15_B, ENS_H15_UNROLL, ENS_H15_THREADS, ENS_H15_MINB, ENS_H15_MAXT)
ENS_SHAPE(16, 5, 4, false, 64, 1)
#undef ENS_SHAPE
#undef ENS_SHAPE_T

// MODE: 0 = fixed step (3 evaluations), 1 = adaptive step, 2 = fixed step with carried a, j (2 evaluations)
template <int N, int MODE>
constexpr auto kernel_ptr() {
    using S = ShapeOf<N>;
    return &hermite_kernel<N, S::L, S::B, S::UNROLL, S::MAXT, S::MINB, MODE == 1, MODE == 2>;
}

template <int N, int MODE>
KernelInfo info_of() {
    using S = ShapeOf<N>;
    KernelInfo k;
    k.fn = (const void*)kernel_ptr<N, MODE>();
    k.shape.L = S::L;
    k.shape.B = S::B;
    k.threads = S::THREADS;
    return k;
}

template <int N, int MODE>
cudaError_t launch_n(const View& v, const StepArgs& a, int threads, cudaStream_t s, int64_t* blocks_out) {
    using S = ShapeOf<N>;
    if (threads > S::MAXT) threads = S::MAXT;  // __launch_bounds__ of the kernel
    const int64_t sys_per_warp = 32 / S::L;
    const int64_t warps = (v.n_sys + sys_per_warp - 1) / sys_per_warp;
    const int wpb = threads / 32;
    int64_t blocks = (warps + wpb - 1) / wpb;
    if constexpr (MODE == 1) {  // persistent grid: what the device holds at once; lane groups pull systems from a.counter
        int dev = 0, sms = 0, per_sm = 0;
        cudaError_t err = cudaGetDevice(&dev);
        if (err == cudaSuccess) err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (err == cudaSuccess)
            err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel_ptr<N, MODE>(), threads, 0);
        if (err != cudaSuccess) return err;
        const int64_t resident = (int64_t)sms * (per_sm > 0 ? per_sm : 1);
        if (blocks > resident) blocks = resident;
    }
    if (blocks_out) *blocks_out = blocks;
    kernel_ptr<N, MODE>()<<<(unsigned)blocks, threads, 0, s>>>(v, a);
    return cudaGetLastError();
}

}  // namespace

#define ENS_FOR_EACH_N(X) X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(11) X(12) X(13) X(14) X(15) X(16)

KernelInfo hermite_kernel_for(int n_body, int mode) {
    switch (n_body) {
#define X(N_) \
    case N_: return mode == 1 ? info_of<N_, 1>() : mode == 2 ? info_of<N_, 2>() : info_of<N_, 0>();
        ENS_FOR_EACH_N(X)
#undef X
    }
    KernelInfo none;
    none.fn = nullptr;
    none.shape.L = none.shape.B = 0;
    none.threads = 0;
    return none;
}

cudaError_t launch_hermite(const View& v, const StepArgs& a, int mode, int threads, cudaStream_t s,
                           int64_t* blocks_out) {
    switch (v.n_body) {
#define X(N_) \
    case N_:  \
        return mode == 1   ? launch_n<N_, 1>(v, a, threads, s, blocks_out) \
               : mode == 2 ? launch_n<N_, 2>(v, a, threads, s, blocks_out) \
                           : launch_n<N_, 0>(v, a, threads, s, blocks_out);
        ENS_FOR_EACH_N(X)
#undef X
    }
    return cudaErrorInvalidValue;
}

namespace {
__global__ void rsqrt_test_kernel(const double* x, double* y, int64_t n) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) y[i] = rsqrt_f64(x[i]);
}
__global__ void rcp_test_kernel(const double* x, double* y, int64_t n) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) y[i] = rcp_f64<true>(x[i]);
}
}  // namespace

}  // namespace ensd

extern "C" ENS_API int ens_test_rsqrt(const double* x, double* y, int64_t n, void* stream) {
    if (!x || !y || n < 0) return ENS_EINVAL;
    if (n == 0) return ENS_OK;
    ensd::rsqrt_test_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(x, y, n);
    return cudaGetLastError() == cudaSuccess ? ENS_OK : ENS_ECUDA;
}

extern "C" ENS_API int ens_test_rcp(const double* x, double* y, int64_t n, void* stream) {
    if (!x || !y || n < 0) return ENS_EINVAL;
    if (n == 0) return ENS_OK;
    ensd::rcp_test_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(x, y, n);
    return cudaGetLastError() == cudaSuccess ? ENS_OK : ENS_ECUDA;
}
