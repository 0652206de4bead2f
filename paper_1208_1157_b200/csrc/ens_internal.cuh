// ens_internal.cuh — types shared by the translation units of libens (CUDA path only; nothing here is used by oracle/).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/ens.h"

namespace ensd {

// Structure-of-arrays ensemble in HBM.  Row r of pos/vel is (body * 3 + component), each row is
// n_pad consecutive systems, so lanes that hold the same body slot of consecutive systems touch consecutive
// addresses (BASELINE.json north_star item 2; the paper's chunked CoalescedStructArray, with the
// chunk taken to be the whole padded ensemble).
struct View {
    double* pos;      // [n_body * 3][n_pad]
    double* vel;      // [n_body * 3][n_pad]
    double* mass;     // [n_body][n_pad]
    double* time;     // [n_pad]
    int32_t* status;  // [n_pad]
    int64_t* nsteps;  // [n_pad]
    int64_t* nreject; // [n_pad] rejected trial steps (adaptive Runge-Kutta)
    int64_t n_sys;
    int64_t n_pad;    // multiple of 64 systems -> every row starts 512-byte aligned
    int n_body;
};

// Arguments of one ens_integrate launch (Alg. 1).
struct StepArgs {
    double dt;
    double t_end;
    double hh;  // dt / 2 (MVS half steps)
    double te;  // t_end folded with the direction of the run: t_end going forward (dt > 0), -t_end going backward
    int64_t max_steps;
    unsigned long long rc2_bits;  // bit pattern of r_close^2 (0 when the monitor is off)
    unsigned long long re2_bits;  // bit pattern of min(r_eject^2, DBL_MAX): also catches inf / NaN positions
    unsigned ce_hi;  // quick test: a body whose three |coordinates| all have a high word below this is inside r_eject
    // MVS quick test (heliocentric Q, centre of mass Xcm): |Q_c| < ce / 4 and |Xcm_c| < ce / 2 bound every barycentric
    // coordinate by ce; a planet with some |Q_c| > r_close is farther than r_close from the star
    unsigned ceq_hi, cex_hi, rc1_hi;
    // Step-size powers of Eq. 3 / Eq. 4 folded into per-launch constants (hermite_kernel.cuh), computed once on the
    // host in IEEE double and read by the kernels straight from the constant bank (no registers held across the loop):
    //   x_p = x + h v + p_a a0 + p_j j0              v_p = v + h a0 + p_a j0
    //   C_x = x + h v + cx_a a0 + cx_j j0            C_v = v + cv_a a0 + cv_j j0
    //   x_c = C_x + kx_a a1 + kx_j j1                v_c = C_v + kv_a a1 + kv_j j1
    double p_a, p_j, cx_a, cx_j, cv_a, cv_j, kx_a, kx_j, kv_a, kv_j;
    unsigned long long* counter;  // persistent kernels: next system / task index to hand out (zeroed before the launch)
    const int32_t* order;         // adaptive kernels: hand-out order (longest expected run first), or nullptr
    // time-sliced fixed-step kernel (hermite_kernel<..., SLICED>): tasks = (warp-group of systems, slice of slice_steps
    // steps), handed out slice-major; slice_done[g] = slices group g has completed (zeroed before the launch)
    int32_t* slice_done;
    int64_t slice_steps, n_slices, n_groups;
    double rk_eps;  // accuracy parameter of the adaptive Runge-Kutta integrator
};

inline void fill_step_constants(StepArgs& a) {
    const double h = a.dt, h2 = h * h, h3 = h2 * h;
    a.p_a = 0.5 * h2;
    a.p_j = h3 / 6.0;
    a.cx_a = 0.35 * h2;
    a.cx_j = 0.05 * h3;
    a.cv_a = 0.5 * h;
    a.cv_j = h2 / 12.0;
    a.kx_a = 0.15 * h2;
    a.kx_j = -h3 / 30.0;
    a.kv_a = 0.5 * h;
    a.kv_j = -h2 / 12.0;
}

// How a system of N bodies is spread over a warp: L lanes per system (odd, so the ring of lanes splits the
// cross pairs evenly), B bodies per lane, L * B >= N (slots beyond N are massless far-away dummies).
struct Shape {
    int L, B;
};

struct KernelInfo {
    const void* fn;
    Shape shape;
    int threads;  // threads per block
    int smem_bytes_per_warp = 0;  // dynamic shared memory the kernel is launched with, per warp of the block
};

// Launch-time choices a test or a measurement may override through ens_test_set_option (0 = the library's default).
struct LaunchTune {
    int threads = 0;             // threads per block
    int adaptive_unordered = 0;  // 1: hand the systems of the adaptive kernels out in index order
    int slice_mode = 0;          // fixed-step Hermite: 0 = library decides, 1 = always time-sliced, 2 = never
    int64_t slice_steps = 0;     // steps per slice
    int slice_warps_per_sm = 0;  // persistent warps per SM of the time-sliced grid
};

// adaptive_order.cu: order[] = system indices sorted by decreasing expected number of adaptive steps
struct OrderBuffers {
    float *key_in = nullptr, *key_out = nullptr;
    int32_t *idx_in = nullptr, *idx_out = nullptr;  // idx_out is the order
    void* tmp = nullptr;
    size_t tmp_bytes = 0;
};
cudaError_t adaptive_order_alloc(int64_t n_sys, OrderBuffers& ob);  // complete or empty
cudaError_t adaptive_order(const View& v, double t_end, OrderBuffers& ob, cudaStream_t s);
void adaptive_order_free(OrderBuffers& ob);

// hermite_*.cu / mvs.cu
KernelInfo hermite_kernel_for(int n_body, int mode);  // mode: 0 fixed step, 1 adaptive, 2 carried a/j
// slice_done: int32 [hermite_slice_groups(n_sys, n_body)] scratch of the time-sliced kernel (or nullptr: never sliced)
int64_t hermite_slice_groups(int64_t n_sys, int n_body);
cudaError_t launch_hermite(const View& v, const StepArgs& a, int mode, const LaunchTune& tune, cudaStream_t s,
                           int64_t* blocks_out, const void** fn_out);
KernelInfo rkck_kernel_for(int n_body, bool adaptive);
cudaError_t launch_rkck(const View& v, const StepArgs& a, bool adaptive, int threads, cudaStream_t s, int64_t* blocks_out);
KernelInfo mvs_kernel_for(int n_body, bool merged);
cudaError_t launch_mvs(const View& v, const StepArgs& a, bool merged, int threads, cudaStream_t s, int64_t* blocks_out);

}  // namespace ensd
