// hermite_static.cu — ens_hermite_static (include/ens.h): the fixed-step Hermite step loop for callers that must not
// allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  The caller owns the ensemble (SoA
// device arrays); the one thing the library has to bring is the scratch of the time-sliced
// persistent grid (hermite_kernel<..., SLICED>: the task counter and one progress word per warp-group of systems), and
// here it lives in a file-scope device array instead of the handle's cudaMalloc'ed buffers.
//
// The array is part of the module image: every GPU that loads libens holds its 256.25 KB until the process exits.  Its
// name in host code is a host-side stand-in, not a device address; the address is looked up once per device with
// cudaGetSymbolAddress (that device current) and cached.  Every call shares the array and finds the last call's
// contents in it: the words a launch uses are cleared on the caller's stream before the kernel, and two calls that
// overlap on the GPU (different streams, no dependency between them) race on it.
#include <atomic>
#include <cfloat>
#include <cmath>
#include <cstring>
#include <mutex>

#include "ens_internal.cuh"

namespace ensd {
int record_cuda_error(cudaError_t err, const char* what);  // ens_api.cu: text for ens_strerror(ENS_ECUDA)
}

namespace {

constexpr size_t COUNTER_BYTES = 256;  // the task counter (8 bytes) in a 256-byte slot of its own
constexpr size_t SCRATCH_BYTES = COUNTER_BYTES + sizeof(int32_t) * (size_t)ENS_STATIC_MAX_GROUPS;

static __device__ __align__(256) unsigned char static_scratch[SCRATCH_BYTES];

constexpr int MAX_DEVICES = 64;
std::atomic<unsigned char*> g_scratch_addr[MAX_DEVICES];  // device address of static_scratch, per device (zero-initialised)
std::mutex g_scratch_mutex;

// Device address of static_scratch on the current device; looked up on the first call per device.
cudaError_t scratch_address(unsigned char** out) {
    int dev = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return err;
    if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
    unsigned char* p = g_scratch_addr[dev].load(std::memory_order_acquire);
    if (!p) {
        std::lock_guard<std::mutex> lock(g_scratch_mutex);
        p = g_scratch_addr[dev].load(std::memory_order_relaxed);
        if (!p) {
            void* q = nullptr;
            if ((err = cudaGetSymbolAddress(&q, static_scratch)) != cudaSuccess) return err;
            p = static_cast<unsigned char*>(q);
            g_scratch_addr[dev].store(p, std::memory_order_release);
        }
    }
    *out = p;
    return cudaSuccess;
}

}  // namespace

extern "C" ENS_API int ens_hermite_static(double* pos, double* vel, const double* mass, double* time, int32_t* status,
                                          int64_t* nsteps, int64_t n_sys, int64_t n_pad, int n_body, double dt,
                                          double t_end, int64_t max_steps, double r_close, double r_eject, void* stream) {
    if (!pos || !vel || !mass || !time || !status || !nsteps) return ENS_EINVAL;
    if (n_sys < 1 || n_pad < n_sys || n_body < 2 || n_body > 16) return ENS_EINVAL;
    if (!(dt != 0.0) || !std::isfinite(dt) || std::isnan(t_end) || max_steps < 0) return ENS_EINVAL;
    if (std::isnan(r_close) || std::isnan(r_eject)) return ENS_EINVAL;
    r_close = r_close > 0.0 ? r_close : 0.0;      // as ens_set_monitors: <= 0 switches a monitor off
    r_eject = r_eject > 0.0 ? r_eject : INFINITY;
    const int64_t groups = ensd::hermite_slice_groups(n_sys, n_body);
    if (groups > ENS_STATIC_MAX_GROUPS) return ENS_ETOOLARGE;
    cudaStream_t s = (cudaStream_t)stream;

    unsigned char* scratch = nullptr;
    cudaError_t err = scratch_address(&scratch);
    if (err != cudaSuccess) return ensd::record_cuda_error(err, "ens_hermite_static: cudaGetSymbolAddress");

    ensd::View v{};
    v.pos = pos;
    v.vel = vel;
    v.mass = const_cast<double*>(mass);  // the step loops only read it
    v.time = time;
    v.status = status;
    v.nsteps = nsteps;
    v.nreject = nullptr;  // (adaptive Runge-Kutta only)
    v.n_sys = n_sys;
    v.n_pad = n_pad;
    v.n_body = n_body;

    // the launch arguments ens_integrate builds for ENS_HERMITE (ens_api.cu), monitors included
    ensd::StepArgs a{};
    a.dt = dt;
    a.t_end = t_end;
    a.hh = 0.5 * dt;
    a.te = dt > 0.0 ? t_end : -t_end;
    a.max_steps = max_steps;
    const double rc2 = r_close * r_close;
    double re2 = r_eject * r_eject;
    if (!(re2 < DBL_MAX)) re2 = DBL_MAX;
    memcpy(&a.rc2_bits, &rc2, 8);
    memcpy(&a.re2_bits, &re2, 8);
    {
        const double ce = std::sqrt(re2 / 3.0);
        unsigned long long b;
        memcpy(&b, &ce, 8);
        a.ce_hi = (unsigned)(b >> 32);
        a.ce_hi = a.ce_hi > 0u ? a.ce_hi - 1u : 0u;
        a.cex_hi = a.ce_hi > 0x00400000u ? a.ce_hi - 0x00100000u : 0u;
        a.ceq_hi = a.ce_hi > 0x00400000u ? a.ce_hi - 0x00200000u : 0u;
        memcpy(&b, &r_close, 8);
        a.rc1_hi = (unsigned)(b >> 32) & 0x7fffffffu;
    }
    ensd::fill_step_constants(a);
    a.counter = reinterpret_cast<unsigned long long*>(scratch);
    a.slice_done = reinterpret_cast<int32_t*>(scratch + COUNTER_BYTES);
    a.order = nullptr;

    // always the time-sliced grid: launch_hermite clears the counter and the `groups` progress words it uses on `s`
    // (cudaMemsetAsync) and launches; with max_steps == 0 it launches the plain kernel, which uses no scratch
    ensd::LaunchTune tune;
    tune.slice_mode = 1;
    err = ensd::launch_hermite(v, a, 0, tune, s, nullptr, nullptr);
    if (err != cudaSuccess) return ensd::record_cuda_error(err, "ens_hermite_static launch");
    return ENS_OK;
}
