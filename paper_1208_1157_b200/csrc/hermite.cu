// hermite.cu — instantiations of the fused Hermite step-loop kernel and the n_body -> (L, B) dispatch.
#include <cmath>

#include "hermite_kernel.cuh"

namespace ensd {

namespace {

// n_body -> lanes per system L (odd), bodies per lane B, L * B >= n_body.  Exact fits for 2-6, 9, 10, 12, 15;
// the others run in the next larger shape with massless dummy slots.  The values are the winners of the sweeps
// recorded in DESIGN.md section 8 (tuning record).
//   UNROLL   1: three inlined copies of the evaluation (straight-line step); 2: two (the corrector iterations are a loop
//            around one); 0: a 3-phase loop around one copy
//   THREADS  threads per block;  MAXT, MINB = __launch_bounds__ (register cap 65536 / (MAXT * MINB))
//   MODE     0 = fixed step (3 evaluations), 1 = adaptive step, 2 = carried a, j (2 evaluations), 3 = MODE 0 time-sliced
template <int N> struct ShapeBase;
#define ENS_SHAPE(N_, L_, B_, UNROLL_, THREADS_, MINB_, MAXT_)                              \
    template <> struct ShapeBase<N_> {                                                      \
        static constexpr int L = L_, B = B_, THREADS = THREADS_, MINB = MINB_, MAXT = MAXT_; \
        static constexpr int UNROLL = UNROLL_;                                              \
    };
// the shape of (N, MODE): the per-N entry unless a mode has its own launch bounds below (L and B never differ by mode)
template <int N, int MODE> struct ShapeOf : ShapeBase<N> {};
#define ENS_SHAPE_MODE(N_, MODE_, UNROLL_, THREADS_, MINB_, MAXT_)                                       \
    template <> struct ShapeOf<N_, MODE_> {                                                              \
        static constexpr int L = ShapeBase<N_>::L, B = ShapeBase<N_>::B, THREADS = THREADS_, MINB = MINB_, \
                             MAXT = MAXT_;                                                               \
        static constexpr int UNROLL = UNROLL_;                                                           \
    };
//        N  L  B  unroll threads minBlocks maxThreads
ENS_SHAPE(2, 1, 2, 1, 64, 1, 128)
// n_body = 3 (config 1, the metric): register cap 128 (125 used, no spills), 8 blocks of 2 warps per SM
ENS_SHAPE(3, 1, 3, 1, 64, 7, 64)
ENS_SHAPE(4, 1, 4, 1, 64, 1, 128)
ENS_SHAPE(5, 1, 5, 1, 64, 1, 128)
// n_body = 6 (config 2): one system per thread, all 15 pairs in one lane, no shuffles: 0.62 of FP64 issue peak against
// 0.54 for the best 3-lane shape; 32-thread blocks spread the 1024 warps of config 2 evenly over the SMs; straight-line
// step 0.668 against 0.653 for the 3-phase loop; with the corrector iterations rolled (24 KB of code per step instead of
// 35 KB) 0.730 against 0.689
ENS_SHAPE(6, 1, 6, 2, 32, 1, 32)
// n_body = 7, 8: still one system per thread.  The state no longer fits 255 registers (336 / 664 B of it live in
// local memory, L1-resident: the step loop touches no other memory), yet every lane does useful work and nothing is
// shuffled: 0.65 / 0.63 of FP64 issue peak against 0.36 / 0.46 for 3 lanes x 3 bodies (9 slots for 7 or 8 bodies).
// From n_body = 9 on the spill traffic wins (0.44 against 0.59) and the lane-split shapes take over.  Two copies of
// the evaluation (rolled corrector iterations) spill less than the 3-phase loop around one (112 / 552 B against
// 336 / 688 B) and are 3 - 4 % faster.
ENS_SHAPE(7, 1, 7, 2, 32, 1, 32)
ENS_SHAPE(8, 1, 8, 2, 32, 1, 32)
// n_body = 9 .. 12: the evaluation of these shapes is small enough (12 / 9 / 22 pairs per lane) for a straight-line step:
// three copies at n = 9, 10 (+5 %, +3 % at 32768 systems; n = 10 at 131072 systems, the paper's largest Table 3 shape:
// 0.617 -> 0.664), two at n = 11, 12 (+2 .. 3 %); the 5 x 3 shapes (n >= 13) stay on the 3-phase loop (three copies:
// 0.54 against 0.64 on config 3)
ENS_SHAPE(9, 3, 3, 1, 64, 1, 128)
// n_body = 10 (the paper's largest Table 3 shape): 168 registers -> 12 warps per SM: 0.60 against 0.54 at 242 registers
ENS_SHAPE(10, 5, 2, 1, 64, 3, 128)
ENS_SHAPE(11, 3, 4, 2, 64, 1, 128)
ENS_SHAPE(12, 3, 4, 2, 64, 1, 128)
ENS_SHAPE(13, 5, 3, 0, 64, 1, 128)
ENS_SHAPE(14, 5, 3, 0, 64, 1, 128)
ENS_SHAPE(15, 5, 3, 0, 64, 1, 128)
ENS_SHAPE(16, 5, 4, 0, 64, 1, 128)
// the carried accelerations and jerks are 18 more live doubles at n_body = 3: 128 registers spilled 120 B of them
ENS_SHAPE_MODE(3, 2, 1, 64, 5, 64)
// n_body = 6 with carried a, j: the straight-line step spilled 464 B; the 3-phase loop spills 16 B and is 3.7 % faster
ENS_SHAPE_MODE(6, 2, 0, 32, 1, 32)
// the adaptive and the 2-evaluation kernels of the many-lane shapes keep the 3-phase loop
ENS_SHAPE_MODE(9, 1, 0, 64, 1, 128)
ENS_SHAPE_MODE(9, 2, 0, 64, 1, 128)
ENS_SHAPE_MODE(10, 1, 0, 64, 3, 128)
ENS_SHAPE_MODE(10, 2, 0, 64, 3, 128)
ENS_SHAPE_MODE(11, 1, 0, 64, 1, 128)
ENS_SHAPE_MODE(11, 2, 0, 64, 1, 128)
ENS_SHAPE_MODE(12, 1, 0, 64, 1, 128)
ENS_SHAPE_MODE(12, 2, 0, 64, 1, 128)
#undef ENS_SHAPE
#undef ENS_SHAPE_MODE

// MODE: 0 = fixed step (3 evaluations), 1 = adaptive step, 2 = fixed step with carried a, j (2 evaluations),
//       3 = MODE 0 on a time-sliced persistent grid (same arithmetic, bit-identical results)
template <int N, int MODE>
constexpr auto kernel_ptr() {
    using S = ShapeOf<N, MODE>;
    return &hermite_kernel<N, S::L, S::B, S::UNROLL, S::MAXT, S::MINB, MODE == 1, MODE == 2, MODE == 3>;
}

template <int N, int MODE>
KernelInfo info_of() {
    using S = ShapeOf<N, MODE>;
    KernelInfo k;
    k.fn = (const void*)kernel_ptr<N, MODE>();
    k.shape.L = S::L;
    k.shape.B = S::B;
    k.threads = S::THREADS;
    k.smem_bytes_per_warp = ring_smem_words<S::L, S::B>() * (int)sizeof(double2);
    return k;
}

// dynamic shared memory of a block of `threads` threads (the cross-lane ring's visitor and return words; 0 for L = 1)
template <int N, int MODE>
constexpr size_t ring_smem_bytes(int threads) {
    using S = ShapeOf<N, MODE>;
    return (size_t)(threads / 32) * ring_smem_words<S::L, S::B>() * sizeof(double2);
}

// blocks of `threads` threads the device holds at once
template <int N, int MODE>
cudaError_t resident_blocks(int threads, int64_t* out) {
    int dev = 0, sms = 0, per_sm = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err == cudaSuccess) err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (err == cudaSuccess) err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel_ptr<N, MODE>(), threads, ring_smem_bytes<N, MODE>(threads));
    *out = (int64_t)sms * (per_sm > 0 ? per_sm : 1);
    return err;
}

template <int N, int MODE>
cudaError_t launch_n(const View& v, StepArgs a, const LaunchTune& tune, cudaStream_t s, int64_t* blocks_out,
                     const void** fn_out) {
    using S = ShapeOf<N, MODE>;
    int threads = tune.threads ? tune.threads : S::THREADS;
    if (threads > S::MAXT) threads = S::MAXT;  // __launch_bounds__ of the kernel
    const int64_t sys_per_warp = 32 / S::L;
    const int64_t warps = (v.n_sys + sys_per_warp - 1) / sys_per_warp;
    const int wpb = threads / 32;
    int64_t blocks = (warps + wpb - 1) / wpb;
    cudaError_t err = cudaSuccess;
    if constexpr (MODE == 1) {  // persistent grid; lane groups pull systems from a.counter
        int64_t resident = 0;  // what the device holds at once
        if ((err = resident_blocks<N, MODE>(threads, &resident)) != cudaSuccess) return err;
        // Systems take different numbers of steps (config 1: the longest 2.2 x the mean), each is a serial chain, and the
        // launch ends with the last one: what counts is systems per lane group (the longest-first hand-out balances only
        // when every group gets several), not resident warps.  Measured: two warps per SM
        // sub-partition are never slower than four (n_body = 3: 131072 systems +11 %, 524288 +1 %); one-system-per-thread
        // shapes with fewer than 1.5 systems per lane of such a grid run faster on one warp per sub-partition (n_body = 3,
        // 32768 systems: +17 %; n_body = 6: +53 %), the many-lane shapes do not (a lone warp cannot hide its ring).
        int dev = 0, sms = 0;
        if ((err = cudaGetDevice(&dev)) != cudaSuccess) return err;
        if ((err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return err;
        const int64_t per_sm = resident / sms;
        const int64_t g = wpb >= 4 ? 1 : 4 / wpb;  // blocks per SM that give every sub-partition one warp
        int64_t k = 2;
        if (S::L == 1 && 2 * v.n_sys < 3 * ((int64_t)sms * 2 * g * threads)) k = 1;
        if (k * g < per_sm) resident = k * g * sms;
        if (blocks > resident) blocks = resident;
    }
    if constexpr (MODE == 0) {
        // Time slicing pays when the ensemble is a few waves of resident warps and the last one is mostly empty: that
        // wave would otherwise run a whole pass on a nearly idle device (config 3: 1.15 waves).  Measured (DESIGN.md
        // section 8): a gain for the many-lane shapes (large state per warp, 2 warps per SM sub-partition); a loss
        // for one-system-per-thread shapes, whose partly filled last wave still saturates the FP64 pipe.
        int64_t resident = 0;
        if ((err = resident_blocks<N, 3>(threads, &resident)) != cudaSuccess) return err;
        if (tune.slice_warps_per_sm > 0) {
            int dev = 0, sms = 0;
            if ((err = cudaGetDevice(&dev)) != cudaSuccess) return err;
            if ((err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return err;
            const int64_t want = ((int64_t)sms * tune.slice_warps_per_sm + wpb - 1) / wpb;
            if (want < resident) resident = want;
        }
        const bool tail = S::L > 1 && blocks > resident && blocks < 4 * resident && 2 * (blocks % resident) < resident;
        const bool sliced = a.slice_done && a.max_steps > 0 &&
                            (tune.slice_mode == 1 || (tune.slice_mode == 0 && tail && a.max_steps >= 256));
        if (sliced) {
            // ~64 slices of the expected run (at least 32 steps each: a slice costs one extra evaluation + load/store)
            double expect = (double)a.max_steps;
            if (std::isfinite(a.t_end)) expect = fmin(expect, ceil(fabs(a.t_end / a.dt)) + 1.0);
            int64_t k = tune.slice_steps > 0 ? tune.slice_steps : (int64_t)ceil(expect / 64.0);
            if (tune.slice_steps <= 0 && k < 32) k = 32;
            if (k > a.max_steps) k = a.max_steps;
            a.slice_steps = k;
            // at most 256 slices: the last one is open-ended (it runs whatever is left of max_steps), so a huge step
            // budget with a time limit (max_steps = 10^9, t_end = 20) does not turn into millions of empty tasks
            a.n_slices = (a.max_steps + k - 1) / k;
            if (a.n_slices > 256) a.n_slices = 256;
            a.n_groups = warps;
            if (blocks > resident) blocks = resident;
            if ((err = cudaMemsetAsync(a.counter, 0, sizeof(unsigned long long), s)) != cudaSuccess) return err;
            if ((err = cudaMemsetAsync(a.slice_done, 0, sizeof(int32_t) * (size_t)warps, s)) != cudaSuccess) return err;
            if (blocks_out) *blocks_out = blocks;
            if (fn_out) *fn_out = (const void*)kernel_ptr<N, 3>();
            kernel_ptr<N, 3>()<<<(unsigned)blocks, threads, ring_smem_bytes<N, 3>(threads), s>>>(v, a);
            return cudaGetLastError();
        }
    }
    if (blocks_out) *blocks_out = blocks;
    if (fn_out) *fn_out = (const void*)kernel_ptr<N, MODE>();
    kernel_ptr<N, MODE>()<<<(unsigned)blocks, threads, ring_smem_bytes<N, MODE>(threads), s>>>(v, a);
    return cudaGetLastError();
}

}  // namespace

#define ENS_FOR_EACH_N(X) X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(11) X(12) X(13) X(14) X(15) X(16)

KernelInfo hermite_kernel_for(int n_body, int mode) {
    switch (n_body) {
#define X(N_) \
    case N_: return mode == 1 ? info_of<N_, 1>() : mode == 2 ? info_of<N_, 2>() : mode == 3 ? info_of<N_, 3>() : info_of<N_, 0>();
        ENS_FOR_EACH_N(X)
#undef X
    }
    KernelInfo none;
    none.fn = nullptr;
    none.shape.L = none.shape.B = 0;
    none.threads = 0;
    return none;
}

cudaError_t launch_hermite(const View& v, const StepArgs& a, int mode, const LaunchTune& tune, cudaStream_t s,
                           int64_t* blocks_out, const void** fn_out) {
    switch (v.n_body) {
#define X(N_) \
    case N_:  \
        return mode == 1   ? launch_n<N_, 1>(v, a, tune, s, blocks_out, fn_out) \
               : mode == 2 ? launch_n<N_, 2>(v, a, tune, s, blocks_out, fn_out) \
                           : launch_n<N_, 0>(v, a, tune, s, blocks_out, fn_out);
        ENS_FOR_EACH_N(X)
#undef X
    }
    return cudaErrorInvalidValue;
}

int64_t hermite_slice_groups(int64_t n_sys, int n_body) {
    switch (n_body) {
#define X(N_) \
    case N_: return (n_sys + 32 / ShapeBase<N_>::L - 1) / (32 / ShapeBase<N_>::L);
        ENS_FOR_EACH_N(X)
#undef X
    }
    return 0;
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
