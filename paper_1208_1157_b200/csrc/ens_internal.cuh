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
    int64_t n_sys;
    int64_t n_pad;    // multiple of 64 systems -> every row starts 512-byte aligned
    int n_body;
};

// Arguments of one ens_integrate launch (Alg. 1).
struct StepArgs {
    double dt;
    double t_end;
    int64_t max_steps;
    unsigned long long rc2_bits;  // bit pattern of r_close^2 (0 when the monitor is off)
    unsigned long long re2_bits;  // bit pattern of min(r_eject^2, DBL_MAX): also catches inf / NaN positions
};

// How a system of N bodies is spread over a warp: L lanes per system (odd, so the ring of lanes splits the
// cross pairs evenly), B bodies per lane, L * B >= N (slots beyond N are massless far-away dummies).
struct Shape {
    int L, B;
};

struct KernelInfo {
    const void* fn;
    Shape shape;
    int threads;  // threads per block
};

// hermite_*.cu / mvs.cu
KernelInfo hermite_kernel_for(int n_body);
cudaError_t launch_hermite(const View& v, const StepArgs& a, int threads, cudaStream_t s, int64_t* blocks_out);
KernelInfo mvs_kernel_for(int n_body);
cudaError_t launch_mvs(const View& v, const StepArgs& a, int threads, cudaStream_t s, int64_t* blocks_out);

}  // namespace ensd
