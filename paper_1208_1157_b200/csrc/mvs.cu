// mvs.cu — instantiations of the fused MVS step-loop kernel and the n_body -> (L, B) dispatch.
#include "mvs_kernel.cuh"

namespace ensd {

namespace {

// n_body -> lanes per system L (odd), planets per lane B, L * B >= n_body - 1 (the star is held by every lane).
template <int N> struct MvsShape;
#define ENS_MVS_SHAPE(N_, L_, B_, THREADS_, MAXREG_)                           \
    template <> struct MvsShape<N_> {                                          \
        static constexpr int L = L_, B = B_, THREADS = THREADS_, MAXREG = MAXREG_; \
    };
//            N   L  B  threads maxRegisters
ENS_MVS_SHAPE(2, 1, 1, 128, 255)
ENS_MVS_SHAPE(3, 1, 2, 128, 255)
// config 4 (3 planets): 64-thread blocks, 168 registers (12 warps per SM): sweeps in DESIGN.md section 8
ENS_MVS_SHAPE(4, 1, 3, 64, 168)
ENS_MVS_SHAPE(5, 1, 4, 128, 255)
ENS_MVS_SHAPE(6, 1, 5, 128, 255)
// n_body = 7 .. 9: one system per thread (up to 376 B of the state in local memory) beats the 3-lane shapes by 11 - 63 %
ENS_MVS_SHAPE(7, 1, 6, 128, 255)
ENS_MVS_SHAPE(8, 1, 7, 128, 255)
ENS_MVS_SHAPE(9, 1, 8, 128, 255)
ENS_MVS_SHAPE(10, 3, 3, 128, 255)
ENS_MVS_SHAPE(11, 5, 2, 128, 255)
ENS_MVS_SHAPE(12, 3, 4, 128, 255)
ENS_MVS_SHAPE(13, 3, 4, 128, 255)
ENS_MVS_SHAPE(14, 5, 3, 128, 255)
ENS_MVS_SHAPE(15, 5, 3, 128, 255)
ENS_MVS_SHAPE(16, 5, 3, 128, 255)
#undef ENS_MVS_SHAPE

template <int N, bool MERGED = false>
constexpr auto kernel_ptr() {
    using S = MvsShape<N>;
    return &mvs_kernel<N, S::L, S::B, S::MAXREG, MERGED>;
}

template <int N, bool MERGED = false>
KernelInfo info_of() {
    using S = MvsShape<N>;
    KernelInfo k;
    k.fn = (const void*)kernel_ptr<N, MERGED>();
    k.shape.L = S::L;
    k.shape.B = S::B;
    k.threads = S::THREADS;
    k.smem_bytes_per_warp = acc_ring_smem_words<S::L, S::B>() * (int)sizeof(double2);
    return k;
}

template <int N, bool MERGED>
cudaError_t launch_n(const View& v, const StepArgs& a, int threads, cudaStream_t s, int64_t* blocks_out) {
    using S = MvsShape<N>;
    if (threads > S::THREADS) threads = S::THREADS;  // __launch_bounds__ of the kernel
    const int64_t sys_per_warp = 32 / S::L;
    const int64_t warps = (v.n_sys + sys_per_warp - 1) / sys_per_warp;
    const int wpb = threads / 32;
    const int64_t blocks = (warps + wpb - 1) / wpb;
    if (blocks_out) *blocks_out = blocks;
    kernel_ptr<N, MERGED>()<<<(unsigned)blocks, threads, (size_t)(threads / 32) * acc_ring_smem_words<S::L, S::B>() * sizeof(double2), s>>>(v, a);
    return cudaGetLastError();
}

}  // namespace

#define ENS_FOR_EACH_N(X) X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(11) X(12) X(13) X(14) X(15) X(16)

KernelInfo mvs_kernel_for(int n_body, bool merged) {
    switch (n_body) {
#define X(N_) \
    case N_: return merged ? info_of<N_, true>() : info_of<N_>();
        ENS_FOR_EACH_N(X)
#undef X
    }
    KernelInfo none;
    none.fn = nullptr;
    none.shape.L = none.shape.B = 0;
    none.threads = 0;
    return none;
}

cudaError_t launch_mvs(const View& v, const StepArgs& a, bool merged, int threads, cudaStream_t s, int64_t* blocks_out) {
    switch (v.n_body) {
#define X(N_) \
    case N_: return merged ? launch_n<N_, true>(v, a, threads, s, blocks_out) : launch_n<N_, false>(v, a, threads, s, blocks_out);
        ENS_FOR_EACH_N(X)
#undef X
    }
    return cudaErrorInvalidValue;
}

}  // namespace ensd
