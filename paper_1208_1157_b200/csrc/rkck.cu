// rkck.cu — instantiations of the fused Cash-Karp step-loop kernel, the n_body -> (L, B) dispatch and the tableau.
#include "rkck_kernel.cuh"

namespace ensd {

namespace {

// n_body -> lanes per system L (odd), bodies per lane B, L * B >= n_body.  Five stage accelerations per body live in
// registers, so a lane holds fewer bodies than in the Hermite kernel.
template <int N> struct RkShape;
// MAXREG_A: register cap of the adaptive kernel (per-system step size, error sums and counters are live on top)
#define ENS_RK_SHAPE_A(N_, L_, B_, THREADS_, MAXREG_, MAXREG_A_)                                         \
    template <> struct RkShape<N_> {                                                                     \
        static constexpr int L = L_, B = B_, THREADS = THREADS_, MAXREG = MAXREG_, MAXREG_A = MAXREG_A_; \
        static constexpr bool ROLLED = (N_ == 6 || N_ == 7) || (L_ == 5 && B_ >= 3) || (L_ == 3 && B_ >= 4); /* stages 2 .. 6 as a loop (rkck_kernel.cuh) */ \
    };
#define ENS_RK_SHAPE(N_, L_, B_, THREADS_, MAXREG_) ENS_RK_SHAPE_A(N_, L_, B_, THREADS_, MAXREG_, MAXREG_)
//           N   L  B  threads maxRegisters
ENS_RK_SHAPE(2, 1, 2, 64, 255)
// n_body = 3 (config 1's ensemble): 168 registers -> 6 blocks of 2 warps per SM, no spills (fixed step)
ENS_RK_SHAPE_A(3, 1, 3, 64, 168, 232)
ENS_RK_SHAPE(4, 1, 4, 64, 255)
// n_body = 5, 7: one system per thread with part of the stage accelerations in local memory (344 / 1448 B, L1-resident)
// beats the padded lane-split shapes: 9.0e9 against 5.0e9 and 2.5e9 against 2.1e9 system-steps/s
ENS_RK_SHAPE(5, 1, 5, 32, 255)
// n_body = 6: one system per thread with the rolled stage loop (864 B of stage accelerations in local memory): 5.63e9
// against 5.30e9 system-steps/s for 3 lanes x 2 bodies
ENS_RK_SHAPE(6, 1, 6, 32, 255)
ENS_RK_SHAPE(7, 1, 7, 32, 255)
ENS_RK_SHAPE(8, 3, 3, 64, 255)
ENS_RK_SHAPE(9, 3, 3, 64, 255)
ENS_RK_SHAPE(10, 5, 2, 64, 255)
// n_body = 11, 12: 3 lanes x 4 bodies (12 slots; the stage accelerations of 4 bodies per lane fit because the rolled stage
// loop keeps them in local memory): 9.2e8 against 6.2e8 / 6.4e8 system-steps/s for 5 x 3 (15 slots)
ENS_RK_SHAPE(11, 3, 4, 64, 255)
ENS_RK_SHAPE(12, 3, 4, 64, 255)
ENS_RK_SHAPE(13, 5, 3, 64, 255)
ENS_RK_SHAPE(14, 5, 3, 64, 255)
ENS_RK_SHAPE(15, 5, 3, 64, 255)
ENS_RK_SHAPE(16, 5, 4, 64, 255)
#undef ENS_RK_SHAPE
#undef ENS_RK_SHAPE_A

template <int N, bool ADAPT = false>
constexpr auto kernel_ptr() {
    using S = RkShape<N>;
    if constexpr (ADAPT)
        return &rkck_adaptive_kernel<N, S::L, S::B, S::MAXREG_A, S::ROLLED>;
    else
        return &rkck_kernel<N, S::L, S::B, S::MAXREG, S::ROLLED>;
}

template <int N, bool ADAPT = false>
KernelInfo info_of() {
    using S = RkShape<N>;
    KernelInfo k;
    k.fn = (const void*)kernel_ptr<N, ADAPT>();
    k.shape.L = S::L;
    k.shape.B = S::B;
    k.threads = S::THREADS;
    k.smem_bytes_per_warp = acc_ring_smem_words<S::L, S::B>() * (int)sizeof(double2);
    return k;
}

// Cash & Karp's tableau (the published rationals) and the products the kernel uses, all formed in long double and
// rounded once.
RkCoef coefficients(double h) {
    typedef long double R;
    const R A[6][5] = {{0, 0, 0, 0, 0},
                       {R(1) / 5, 0, 0, 0, 0},
                       {R(3) / 40, R(9) / 40, 0, 0, 0},
                       {R(3) / 10, R(-9) / 10, R(6) / 5, 0, 0},
                       {R(-11) / 54, R(5) / 2, R(-70) / 27, R(35) / 27, 0},
                       {R(1631) / 55296, R(175) / 512, R(575) / 13824, R(44275) / 110592, R(253) / 4096}};
    const R b[6] = {R(37) / 378, 0, R(250) / 621, R(125) / 594, 0, R(512) / 1771};
    RkCoef q;
    const R H = h, H2 = H * H;
    for (int i = 0; i < 6; ++i) {
        R c = 0;
        for (int j = 0; j < i; ++j) c += A[i][j];
        q.ch[i] = (double)(c * H);
        q.hb[i] = (double)(b[i] * H);
        for (int ll = 0; ll < 4; ++ll) {
            R s = 0;
            for (int j = ll + 1; j < i; ++j) s += A[i][j] * A[j][ll];
            q.h2AA[i][ll] = (double)(s * H2);
        }
    }
    for (int ll = 0; ll < 5; ++ll) {
        R s = 0;
        for (int i = ll + 1; i < 6; ++i) s += b[i] * A[i][ll];
        q.h2bA[ll] = (double)(s * H2);
    }
    return q;
}

// the same tableau without the powers of h, plus the weights of the embedded error estimate d = b5 - b4 (adaptive kernel)
RkUnit unit_coefficients() {
    typedef long double R;
    const R A[6][5] = {{0, 0, 0, 0, 0},
                       {R(1) / 5, 0, 0, 0, 0},
                       {R(3) / 40, R(9) / 40, 0, 0, 0},
                       {R(3) / 10, R(-9) / 10, R(6) / 5, 0, 0},
                       {R(-11) / 54, R(5) / 2, R(-70) / 27, R(35) / 27, 0},
                       {R(1631) / 55296, R(175) / 512, R(575) / 13824, R(44275) / 110592, R(253) / 4096}};
    const R b5[6] = {R(37) / 378, 0, R(250) / 621, R(125) / 594, 0, R(512) / 1771};
    const R b4[6] = {R(2825) / 27648, 0, R(18575) / 48384, R(13525) / 55296, R(277) / 14336, R(1) / 4};
    RkUnit q;
    for (int i = 0; i < 6; ++i) {
        R c = 0;
        for (int j = 0; j < i; ++j) c += A[i][j];
        q.c[i] = (double)c;
        q.b[i] = (double)b5[i];
        q.d[i] = (double)(b5[i] - b4[i]);
        for (int ll = 0; ll < 4; ++ll) {
            R s = 0;
            for (int j = ll + 1; j < i; ++j) s += A[i][j] * A[j][ll];
            q.AA[i][ll] = (double)s;
        }
    }
    for (int ll = 0; ll < 5; ++ll) {
        R s = 0, sd = 0;
        for (int i = ll + 1; i < 6; ++i) {
            s += b5[i] * A[i][ll];
            sd += (b5[i] - b4[i]) * A[i][ll];
        }
        q.bA[ll] = (double)s;
        q.dA[ll] = (double)sd;
    }
    return q;
}

template <int N>
cudaError_t launch_adaptive_n(const View& v, const StepArgs& a, int threads, cudaStream_t s, int64_t* blocks_out) {
    using S = RkShape<N>;
    if (threads > S::THREADS) threads = S::THREADS;
    const int64_t sys_per_warp = 32 / S::L;
    const int64_t warps = (v.n_sys + sys_per_warp - 1) / sys_per_warp;
    const int wpb = threads / 32;
    int64_t blocks = (warps + wpb - 1) / wpb;
    int dev = 0, sms = 0, per_sm = 0;  // persistent grid: what the device holds at once
    cudaError_t err = cudaGetDevice(&dev);
    if (err == cudaSuccess) err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (err == cudaSuccess) err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel_ptr<N, true>(), threads, (size_t)(threads / 32) * acc_ring_smem_words<S::L, S::B>() * sizeof(double2));
    if (err != cudaSuccess) return err;
    const int64_t resident = (int64_t)sms * (per_sm > 0 ? per_sm : 1);
    if (blocks > resident) blocks = resident;
    if (blocks_out) *blocks_out = blocks;
    kernel_ptr<N, true>()<<<(unsigned)blocks, threads, (size_t)(threads / 32) * acc_ring_smem_words<S::L, S::B>() * sizeof(double2), s>>>(v, a, unit_coefficients());
    return cudaGetLastError();
}

template <int N>
cudaError_t launch_n(const View& v, const StepArgs& a, int threads, cudaStream_t s, int64_t* blocks_out) {
    using S = RkShape<N>;
    if (threads > S::THREADS) threads = S::THREADS;  // blocks must not exceed 65536 / MAXREG threads
    const int64_t sys_per_warp = 32 / S::L;
    const int64_t warps = (v.n_sys + sys_per_warp - 1) / sys_per_warp;
    const int wpb = threads / 32;
    const int64_t blocks = (warps + wpb - 1) / wpb;
    if (blocks_out) *blocks_out = blocks;
    kernel_ptr<N>()<<<(unsigned)blocks, threads, (size_t)(threads / 32) * acc_ring_smem_words<S::L, S::B>() * sizeof(double2), s>>>(v, a, coefficients(a.dt));
    return cudaGetLastError();
}

}  // namespace

#define ENS_FOR_EACH_N(X) X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(11) X(12) X(13) X(14) X(15) X(16)

KernelInfo rkck_kernel_for(int n_body, bool adaptive) {
    switch (n_body) {
#define X(N_) \
    case N_: return adaptive ? info_of<N_, true>() : info_of<N_>();
        ENS_FOR_EACH_N(X)
#undef X
    }
    KernelInfo none;
    none.fn = nullptr;
    none.shape.L = none.shape.B = 0;
    none.threads = 0;
    return none;
}

cudaError_t launch_rkck(const View& v, const StepArgs& a, bool adaptive, int threads, cudaStream_t s, int64_t* blocks_out) {
    switch (v.n_body) {
#define X(N_) \
    case N_: return adaptive ? launch_adaptive_n<N_>(v, a, threads, s, blocks_out) : launch_n<N_>(v, a, threads, s, blocks_out);
        ENS_FOR_EACH_N(X)
#undef X
    }
    return cudaErrorInvalidValue;
}

}  // namespace ensd
