// ens_api.cu — the C ABI of include/ens.h: handle, SoA buffers, AoS<->SoA transposition, energy, helpers.
// All arithmetic of the method lives in hermite_kernel.cuh / mvs_kernel.cuh; nothing here calls oracle/ and there is
// no CPU fallback: without a device every call that needs one returns ENS_ECUDA.
#include <cfloat>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include "ens_internal.cuh"

namespace {

thread_local char g_cuda_err[256] = "no CUDA error recorded";

int cuda_fail(cudaError_t err, const char* what) {
    snprintf(g_cuda_err, sizeof g_cuda_err, "CUDA error in %s: %s", what, cudaGetErrorString(err));
    (void)cudaGetLastError();  // clear the sticky-less error state
    return err == cudaErrorMemoryAllocation ? ENS_ENOMEM : ENS_ECUDA;
}
#define CU(call)                                            \
    do {                                                    \
        cudaError_t err__ = (call);                         \
        if (err__ != cudaSuccess) return cuda_fail(err__, #call); \
    } while (0)

}  // namespace

namespace ensd {
// for the translation units that hold other entry points (hermite_static.cu): same error text channel
int record_cuda_error(cudaError_t err, const char* what) { return cuda_fail(err, what); }
}  // namespace ensd

namespace {

constexpr int TILE = 64;  // systems per transposition tile = padding granule of the SoA rows

// ---------------------------------------------------------------------------------------------------------------
// AoS [n_sys][K] <-> SoA [K][n_pad] transposition through shared memory, 128-bit global accesses on both sides
// (north_star item 2).  One block per tile of 64 systems; K = 3 n_body (pos, vel) or n_body (mass) is a compile-time
// constant (the index arithmetic of a run-time K made these kernels ALU-bound).  ens_set_state is ONE launch: pos, vel
// and mass tiles one after the other through the same shared buffer, then the time / status / nsteps reset of the
// tile's systems.  Pure data movement: HBM-bound, 16 bytes of traffic per double.
// ---------------------------------------------------------------------------------------------------------------
// the four halves of a transposition; the callers place the __syncthreads between a load and its store
template <int K>
__device__ __forceinline__ void aos_to_tile(const double* __restrict__ src, double* tile, int64_t sys0, int nv,
                                            bool vec_ok) {
    constexpr int Kp = K | 1;  // odd pitch: conflict-free column accesses
    const int total = nv * K;
    const double* s = src + sys0 * K;
    if (vec_ok && (total & 1) == 0) {
        const double2* s2 = reinterpret_cast<const double2*>(s);
#pragma unroll 2
        for (int i = threadIdx.x; i < total / 2; i += blockDim.x) {
            const double2 w = s2[i];
            const int i0 = 2 * i, i1 = 2 * i + 1;
            tile[(i0 / K) * Kp + (i0 % K)] = w.x;
            tile[(i1 / K) * Kp + (i1 % K)] = w.y;
        }
    } else {
        for (int i = threadIdx.x; i < total; i += blockDim.x) tile[(i / K) * Kp + (i % K)] = s[i];
    }
}

template <int K>
__device__ __forceinline__ void tile_to_soa(const double* tile, double* __restrict__ dst, int64_t sys0, int nv,
                                            int64_t n_pad) {
    constexpr int Kp = K | 1;
    // rows of the SoA: two consecutive systems per thread (sys0 and n_pad are multiples of 64: 16-byte aligned)
    for (int i = threadIdx.x; i < K * (TILE / 2); i += blockDim.x) {
        const int k = i / (TILE / 2), sp = (i % (TILE / 2)) * 2;
        double2 w;
        w.x = sp < nv ? tile[sp * Kp + k] : 0.0;
        w.y = sp + 1 < nv ? tile[(sp + 1) * Kp + k] : 0.0;
        *reinterpret_cast<double2*>(dst + (int64_t)k * n_pad + sys0 + sp) = w;
    }
}

template <int K>
__device__ __forceinline__ void soa_to_tile(const double* __restrict__ src, double* tile, int64_t sys0, int64_t n_pad) {
    constexpr int Kp = K | 1;
#pragma unroll 2
    for (int i = threadIdx.x; i < K * (TILE / 2); i += blockDim.x) {
        const int k = i / (TILE / 2), sp = (i % (TILE / 2)) * 2;
        const double2 w = *reinterpret_cast<const double2*>(src + (int64_t)k * n_pad + sys0 + sp);
        tile[sp * Kp + k] = w.x;
        tile[(sp + 1) * Kp + k] = w.y;
    }
}

template <int K>
__device__ __forceinline__ void tile_to_aos(const double* tile, double* __restrict__ dst, int64_t sys0, int nv,
                                            bool vec_ok) {
    constexpr int Kp = K | 1;
    const int total = nv * K;
    double* d = dst + sys0 * K;
    if (vec_ok && (total & 1) == 0) {
        double2* d2 = reinterpret_cast<double2*>(d);
        for (int i = threadIdx.x; i < total / 2; i += blockDim.x) {
            const int i0 = 2 * i, i1 = 2 * i + 1;
            double2 w;
            w.x = tile[(i0 / K) * Kp + (i0 % K)];
            w.y = tile[(i1 / K) * Kp + (i1 % K)];
            d2[i] = w;
        }
    } else {
        for (int i = threadIdx.x; i < total; i += blockDim.x) d[i] = tile[(i / K) * Kp + (i % K)];
    }
}

// pos, vel and mass tiles are in flight together (three shared buffers, one barrier) when they fit 48 KB, else one
// after the other through one buffer
template <int NB>
__global__ void __launch_bounds__(256) pack_state_kernel(const double* __restrict__ pos, const double* __restrict__ vel,
                                                         const double* __restrict__ mass,
                                                         const double* __restrict__ time_src, ensd::View e,
                                                         int vec_pos, int vec_vel, int vec_mass) {
    constexpr int T3 = TILE * ((3 * NB) | 1), T1 = TILE * (NB | 1);
    constexpr bool TOGETHER = (2 * T3 + T1) * sizeof(double) <= 48 * 1024;
    __shared__ double tile[TOGETHER ? 2 * T3 + T1 : T3];
    const int64_t sys0 = (int64_t)blockIdx.x * TILE;
    const int nv = (int)((e.n_sys - sys0 < TILE) ? (e.n_sys - sys0) : TILE);
    if constexpr (TOGETHER) {
        aos_to_tile<3 * NB>(pos, tile, sys0, nv, vec_pos);
        aos_to_tile<3 * NB>(vel, tile + T3, sys0, nv, vec_vel);
        aos_to_tile<NB>(mass, tile + 2 * T3, sys0, nv, vec_mass);
        __syncthreads();
        tile_to_soa<3 * NB>(tile, e.pos, sys0, nv, e.n_pad);
        tile_to_soa<3 * NB>(tile + T3, e.vel, sys0, nv, e.n_pad);
        tile_to_soa<NB>(tile + 2 * T3, e.mass, sys0, nv, e.n_pad);
    } else {
        aos_to_tile<3 * NB>(pos, tile, sys0, nv, vec_pos);
        __syncthreads();
        tile_to_soa<3 * NB>(tile, e.pos, sys0, nv, e.n_pad);
        __syncthreads();
        aos_to_tile<3 * NB>(vel, tile, sys0, nv, vec_vel);
        __syncthreads();
        tile_to_soa<3 * NB>(tile, e.vel, sys0, nv, e.n_pad);
        __syncthreads();
        aos_to_tile<NB>(mass, tile, sys0, nv, vec_mass);
        __syncthreads();
        tile_to_soa<NB>(tile, e.mass, sys0, nv, e.n_pad);
    }
    if (threadIdx.x < TILE) {  // resets the padding systems of the last tile too
        const int64_t i = sys0 + threadIdx.x;
        e.time[i] = (threadIdx.x < nv && time_src) ? time_src[i] : 0.0;
        e.status[i] = ENS_ACTIVE;
        e.nsteps[i] = 0;
        e.nreject[i] = 0;
    }
}

// pos and / or vel (a NULL destination is skipped), plus the per-system rows time / status / nsteps (NULL: skipped)
template <int NB>
__global__ void __launch_bounds__(256) unpack_state_kernel(ensd::View e, double* __restrict__ pos,
                                                           double* __restrict__ vel, double* __restrict__ time,
                                                           int32_t* __restrict__ status, int64_t* __restrict__ nsteps,
                                                           int vec_pos, int vec_vel) {
    constexpr int T3 = TILE * ((3 * NB) | 1);
    constexpr bool TOGETHER = 2 * T3 * sizeof(double) <= 48 * 1024;
    __shared__ double tile[TOGETHER ? 2 * T3 : T3];
    const int64_t sys0 = (int64_t)blockIdx.x * TILE;
    const int nv = (int)((e.n_sys - sys0 < TILE) ? (e.n_sys - sys0) : TILE);
    if (threadIdx.x < nv) {
        const int64_t i = sys0 + threadIdx.x;
        if (time) time[i] = e.time[i];
        if (status) status[i] = e.status[i];
        if (nsteps) nsteps[i] = e.nsteps[i];
    }
    if (TOGETHER && pos && vel) {
        soa_to_tile<3 * NB>(e.pos, tile, sys0, e.n_pad);
        soa_to_tile<3 * NB>(e.vel, tile + (TOGETHER ? T3 : 0), sys0, e.n_pad);
        __syncthreads();
        tile_to_aos<3 * NB>(tile, pos, sys0, nv, vec_pos);
        tile_to_aos<3 * NB>(tile + (TOGETHER ? T3 : 0), vel, sys0, nv, vec_vel);
    } else {
        if (pos) {
            soa_to_tile<3 * NB>(e.pos, tile, sys0, e.n_pad);
            __syncthreads();
            tile_to_aos<3 * NB>(tile, pos, sys0, nv, vec_pos);
            __syncthreads();
        }
        if (vel) {
            soa_to_tile<3 * NB>(e.vel, tile, sys0, e.n_pad);
            __syncthreads();
            tile_to_aos<3 * NB>(tile, vel, sys0, nv, vec_vel);
        }
    }
}

#define ENS_FOR_EACH_NB(X) X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(11) X(12) X(13) X(14) X(15) X(16)

cudaError_t launch_pack(const double* pos, const double* vel, const double* mass, const double* time_src,
                        const ensd::View& v, cudaStream_t s) {
    const unsigned g = (unsigned)(v.n_pad / TILE);
    auto al = [](const void* p) { return (int)((reinterpret_cast<uintptr_t>(p) & 15) == 0); };
    switch (v.n_body) {
#define X(N_) \
    case N_: pack_state_kernel<N_><<<g, 256, 0, s>>>(pos, vel, mass, time_src, v, al(pos), al(vel), al(mass)); break;
        ENS_FOR_EACH_NB(X)
#undef X
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t launch_unpack(const ensd::View& v, double* pos, double* vel, double* time, int32_t* status,
                          int64_t* nsteps, cudaStream_t s) {
    const unsigned g = (unsigned)(v.n_pad / TILE);
    auto al = [](const void* p) { return (int)((reinterpret_cast<uintptr_t>(p) & 15) == 0); };
    switch (v.n_body) {
#define X(N_) \
    case N_: unpack_state_kernel<N_><<<g, 256, 0, s>>>(v, pos, vel, time, status, nsteps, al(pos), al(vel)); break;
        ENS_FOR_EACH_NB(X)
#undef X
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------------
// Energy and angular momentum, Eq. 6 with each unordered pair once (R9).  One thread per system reading
// the SoA rows (coalesced); correctly rounded sqrt and divide.  HBM-bound: (7 n_body + 4) * 8 bytes per system.
// ---------------------------------------------------------------------------------------------------------------
template <int NB>
__global__ void __launch_bounds__(128) energy_kernel(ensd::View e, double* __restrict__ E, double* __restrict__ Lout) {
    const int64_t sys = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (sys >= e.n_sys) return;
    double x[NB][3], m[NB];  // compile-time body count: registers, not local memory
    double ke = 0.0, pe = 0.0, L[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int i = 0; i < NB; ++i) {
        double v[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            x[i][c] = e.pos[(int64_t)(i * 3 + c) * e.n_pad + sys];
            v[c] = e.vel[(int64_t)(i * 3 + c) * e.n_pad + sys];
        }
        m[i] = e.mass[(int64_t)i * e.n_pad + sys];
        ke += 0.5 * m[i] * (v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
        L[0] += m[i] * (x[i][1] * v[2] - x[i][2] * v[1]);
        L[1] += m[i] * (x[i][2] * v[0] - x[i][0] * v[2]);
        L[2] += m[i] * (x[i][0] * v[1] - x[i][1] * v[0]);
    }
#pragma unroll
    for (int i = 0; i < NB; ++i)
#pragma unroll
        for (int k = i + 1; k < NB; ++k) {
            const double dx = x[k][0] - x[i][0], dy = x[k][1] - x[i][1], dz = x[k][2] - x[i][2];
            pe -= m[i] * m[k] / sqrt(dx * dx + dy * dy + dz * dz);
        }
    E[sys] = ke + pe;
    if (Lout) {
        Lout[3 * sys + 0] = L[0];
        Lout[3 * sys + 1] = L[1];
        Lout[3 * sys + 2] = L[2];
    }
}

// ---------------------------------------------------------------------------------------------------------------
// FP64 pipe microbenchmark: 8 independent DFMA chains per thread (MEASURED_PEAKS.json has no FP64
// entry, so the denominator of "% of FP64 peak" is measured here).
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dfma_kernel(int64_t iters, double seed, double* out) {
    double a0 = seed, a1 = seed + 1, a2 = seed + 2, a3 = seed + 3, a4 = seed + 4, a5 = seed + 5, a6 = seed + 6,
           a7 = seed + 7;
    const double b = 0.999999, c = 1e-9;
    for (int64_t i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            a0 = fma(a0, b, c); a1 = fma(a1, b, c); a2 = fma(a2, b, c); a3 = fma(a3, b, c);
            a4 = fma(a4, b, c); a5 = fma(a5, b, c); a6 = fma(a6, b, c); a7 = fma(a7, b, c);
        }
    }
    const double r = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (r == 12345.678) out[0] = r;  // never true; keeps the chains alive
}


// ---------------------------------------------------------------------------------------------------------------
// State log ("the system's current state is written to a buffer in the GPU global device memory"; reading
// R-L1/R-L2 of DESIGN.md).  Runs on the stream between two segments of ens_integrate_logged: every system that
// advanced since its last record (and that the selection asks for) appends one record at an atomic cursor.
// Record r: sys[r], nsteps[r], time[r], status[r], pos[r][n_body][3], vel[r][n_body][3].  HBM-bound data movement.
// ---------------------------------------------------------------------------------------------------------------
struct LogView {
    int64_t capacity;
    unsigned long long* cursor;  // [0] = records appended (may exceed capacity: the excess was dropped)
    int64_t* last;               // [n_pad] nsteps at the last record of each system (-1 = never)
    int64_t *sys, *nsteps;
    double* time;
    int32_t* status;
    double *pos, *vel;
};

__global__ void __launch_bounds__(128) log_kernel(ensd::View e, LogView g, int what) {
    const int64_t sys = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (sys >= e.n_sys) return;
    const int64_t ns = e.nsteps[sys];
    if (ns == g.last[sys]) return;  // nothing new since its last record
    const int st = e.status[sys];
    const bool stopped = st >= ENS_STOP_CLOSE;
    if (!((what & ENS_LOG_SNAPSHOTS) || ((what & ENS_LOG_STOPS) && stopped))) return;
    g.last[sys] = ns;
    const unsigned long long r = atomicAdd(g.cursor, 1ull);
    if ((int64_t)r >= g.capacity) return;  // dropped (counted by the cursor)
    g.sys[r] = sys;
    g.nsteps[r] = ns;
    g.time[r] = e.time[sys];
    g.status[r] = st;
    const int n3 = e.n_body * 3;
    for (int k = 0; k < n3; ++k) {
        g.pos[r * n3 + k] = e.pos[(int64_t)k * e.n_pad + sys];
        g.vel[r * n3 + k] = e.vel[(int64_t)k * e.n_pad + sys];
    }
}

__global__ void log_reset_kernel(int64_t* last, int64_t n, unsigned long long* cursor) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) last[i] = -1;
    if (i == 0) *cursor = 0ull;
}

}  // namespace

struct ens {
    ensd::View v{};
    double r_close = 0.0, r_eject = INFINITY;
    double rk_eps = 1e-9;
    bool have_state = false;
    int device = 0;
    // device staging (AoS) for host-space calls, allocated by the first host-space call (which waits for the stream
    // anyway) or ahead of time by ens_reserve_host_staging
    // (a lazily filled cache: the read-only calls may fill it too, hence mutable)
    mutable double* stage = nullptr;        // [n_sys * n_body * 7] : pos | vel | mass
    mutable double* stage_small = nullptr;  // [n_sys * 4] : time / E | L
    ensd::KernelInfo hermite{}, hermite_sliced{}, hermite_adaptive{}, hermite_carry{}, rkck{}, rkck_adaptive{}, mvs{}, mvs_merged{};
    unsigned long long* counter = nullptr;  // work counter of the persistent kernels
    int32_t* slice_done = nullptr;          // per warp-group slice counters of the time-sliced Hermite kernel
    ensd::OrderBuffers order;               // hand-out order of the adaptive kernels (allocated by ens_create)
    ensd::LaunchTune tune;                  // ens_test_set_option
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    LogView log{};  // capacity 0 = no log buffer
    // bookkeeping that the read-only calls (ens_get_state, ens_energy) update too
    mutable int64_t last_blocks = 0;
    mutable const void* last_fn = nullptr;
    mutable int64_t launches = 0;
    mutable bool timed = false;
};

namespace {

// Every entry point runs on the device the handle was created on, whatever device is current in the calling thread,
// and leaves the caller's current device as it found it.
class DeviceGuard {
  public:
    explicit DeviceGuard(int want) {
        if (cudaGetDevice(&prev_) != cudaSuccess) { err_ = cudaGetLastError(); return; }
        if (prev_ != want) {
            err_ = cudaSetDevice(want);
            switched_ = err_ == cudaSuccess;
        }
    }
    ~DeviceGuard() {
        if (switched_) cudaSetDevice(prev_);
    }
    cudaError_t error() const { return err_; }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;

  private:
    int prev_ = 0;
    bool switched_ = false;
    cudaError_t err_ = cudaSuccess;
};
#define ENS_ON_DEVICE(e)                 \
    DeviceGuard guard__((e)->device);    \
    CU(guard__.error())

int ensure_stage(const ens* e) {
    const int64_t n = e->v.n_sys, nb = e->v.n_body;
    if (!e->stage) CU(cudaMalloc(&e->stage, sizeof(double) * n * nb * 7));
    if (!e->stage_small) CU(cudaMalloc(&e->stage_small, sizeof(double) * n * 4));
    return ENS_OK;
}


}  // namespace

extern "C" {

const char* ens_strerror(int code) {
    switch (code) {
        case ENS_OK: return "ok";
        case ENS_EINVAL: return "invalid argument";
        case ENS_ENOMEM: return "out of device memory";
        case ENS_ECUDA: return g_cuda_err;
        case ENS_ESTATE: return "no state set (call ens_set_state first)";
        case ENS_EUNSUPPORTED: return "unsupported configuration";
        case ENS_ETOOLARGE:
            return "ensemble too large for the static scratch (ens_hermite_static: more than ENS_STATIC_MAX_GROUPS = 65536 "
                   "warp-groups of systems; use a handle, ens_create + ens_integrate)";
        default: return "unknown error code";
    }
}

int ens_create(int64_t n_sys, int n_body, ens_t** out) {
    if (!out) return ENS_EINVAL;
    *out = nullptr;
    if (n_sys < 1 || n_body < 2 || n_body > 16) return ENS_EINVAL;
    int dev = 0;
    CU(cudaGetDevice(&dev));
    ens* e = new (std::nothrow) ens();
    if (!e) return ENS_ENOMEM;
    e->device = dev;
    e->v.n_sys = n_sys;
    e->v.n_body = n_body;
    e->v.n_pad = (n_sys + TILE - 1) / TILE * TILE;
    const int64_t np = e->v.n_pad;
    cudaError_t err = cudaSuccess;
    auto alloc = [&](void** p, size_t bytes) {
        if (err == cudaSuccess) err = cudaMalloc(p, bytes);
    };
    alloc((void**)&e->v.pos, sizeof(double) * np * n_body * 3);
    alloc((void**)&e->v.vel, sizeof(double) * np * n_body * 3);
    alloc((void**)&e->v.mass, sizeof(double) * np * n_body);
    alloc((void**)&e->v.time, sizeof(double) * np);
    alloc((void**)&e->v.status, sizeof(int32_t) * np);
    alloc((void**)&e->v.nsteps, sizeof(int64_t) * np);
    alloc((void**)&e->v.nreject, sizeof(int64_t) * np);
    alloc((void**)&e->counter, sizeof(unsigned long long));
    alloc((void**)&e->slice_done, sizeof(int32_t) * (size_t)ensd::hermite_slice_groups(n_sys, n_body));
    // everything ens_integrate needs is allocated here: device-space calls only enqueue
    if (err == cudaSuccess && n_sys <= 0x7fffffff) err = ensd::adaptive_order_alloc(n_sys, e->order);
    if (err == cudaSuccess) err = cudaEventCreate(&e->ev0);
    if (err == cudaSuccess) err = cudaEventCreate(&e->ev1);
    if (err != cudaSuccess) {
        const int rc = cuda_fail(err, "ens_create");
        ens_destroy(e);
        return rc;
    }
    e->hermite = ensd::hermite_kernel_for(n_body, 0);
    e->hermite_adaptive = ensd::hermite_kernel_for(n_body, 1);
    e->hermite_carry = ensd::hermite_kernel_for(n_body, 2);
    e->hermite_sliced = ensd::hermite_kernel_for(n_body, 3);
    e->rkck = ensd::rkck_kernel_for(n_body, false);
    e->rkck_adaptive = ensd::rkck_kernel_for(n_body, true);
    e->mvs = ensd::mvs_kernel_for(n_body, false);
    e->mvs_merged = ensd::mvs_kernel_for(n_body, true);
    *out = e;
    return ENS_OK;
}

int ens_destroy(ens_t* e) {
    if (!e) return ENS_OK;
    {
        DeviceGuard guard(e->device);
        cudaDeviceSynchronize();
        cudaFree(e->v.pos);
        cudaFree(e->v.vel);
        cudaFree(e->v.mass);
        cudaFree(e->v.time);
        cudaFree(e->v.status);
        cudaFree(e->v.nsteps);
        cudaFree(e->v.nreject);
        cudaFree(e->counter);
        cudaFree(e->slice_done);
        cudaFree(e->log.cursor);
        cudaFree(e->log.last);
        cudaFree(e->log.sys);
        cudaFree(e->log.nsteps);
        cudaFree(e->log.time);
        cudaFree(e->log.status);
        cudaFree(e->log.pos);
        cudaFree(e->log.vel);
        ensd::adaptive_order_free(e->order);
        cudaFree(e->stage);
        cudaFree(e->stage_small);
        if (e->ev0) cudaEventDestroy(e->ev0);
        if (e->ev1) cudaEventDestroy(e->ev1);
        (void)cudaGetLastError();
    }
    delete e;
    return ENS_OK;
}

int ens_reserve_host_staging(ens_t* e) {
    if (!e) return ENS_EINVAL;
    ENS_ON_DEVICE(e);
    return ensure_stage(e);
}

int ens_set_monitors(ens_t* e, double r_close, double r_eject) {
    if (!e || std::isnan(r_close) || std::isnan(r_eject)) return ENS_EINVAL;
    e->r_close = r_close > 0.0 ? r_close : 0.0;
    e->r_eject = r_eject > 0.0 ? r_eject : INFINITY;
    return ENS_OK;
}

int ens_set_rk_tolerance(ens_t* e, double eps) {
    if (!e || !(eps > 0.0) || !std::isfinite(eps)) return ENS_EINVAL;
    e->rk_eps = eps;
    return ENS_OK;
}

int ens_get_rejected(const ens_t* e, int64_t* nreject, int memspace, void* stream) {
    if (!e || !nreject || (memspace != ENS_HOST && memspace != ENS_DEVICE)) return ENS_EINVAL;
    if (!e->have_state) return ENS_ESTATE;
    ENS_ON_DEVICE(e);
    cudaStream_t s = (cudaStream_t)stream;
    CU(cudaMemcpyAsync(nreject, e->v.nreject, sizeof(int64_t) * e->v.n_sys,
                       memspace == ENS_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, s));
    if (memspace == ENS_HOST) CU(cudaStreamSynchronize(s));
    return ENS_OK;
}

int ens_set_state(ens_t* e, const double* pos, const double* vel, const double* mass, const double* time, int memspace,
                  void* stream) {
    if (!e || !pos || !vel || !mass || (memspace != ENS_HOST && memspace != ENS_DEVICE)) return ENS_EINVAL;
    ENS_ON_DEVICE(e);
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t n = e->v.n_sys, nb = e->v.n_body;
    const double *dpos = pos, *dvel = vel, *dmass = mass, *dtime = time;
    if (memspace == ENS_HOST) {
        const int rc = ensure_stage(e);
        if (rc) return rc;
        double* st = e->stage;
        CU(cudaMemcpyAsync(st, pos, sizeof(double) * n * nb * 3, cudaMemcpyHostToDevice, s));
        CU(cudaMemcpyAsync(st + n * nb * 3, vel, sizeof(double) * n * nb * 3, cudaMemcpyHostToDevice, s));
        CU(cudaMemcpyAsync(st + n * nb * 6, mass, sizeof(double) * n * nb, cudaMemcpyHostToDevice, s));
        dpos = st;
        dvel = st + n * nb * 3;
        dmass = st + n * nb * 6;
        if (time) {
            CU(cudaMemcpyAsync(e->stage_small, time, sizeof(double) * n, cudaMemcpyHostToDevice, s));
            dtime = e->stage_small;
        }
    }
    CU(launch_pack(dpos, dvel, dmass, dtime, e->v, s));
    e->launches += 1;
    if (e->log.capacity)  // step counters restart at 0: forget what was logged (records already taken stay)
        CU(cudaMemsetAsync(e->log.last, 0xFF, sizeof(int64_t) * e->v.n_pad, s));
    if (memspace == ENS_HOST) CU(cudaStreamSynchronize(s));
    e->have_state = true;
    return ENS_OK;
}

int ens_integrate(ens_t* e, int integrator, double dt, double t_end, int64_t max_steps, void* stream) {
    if (!e || integrator < ENS_HERMITE || integrator > ENS_RKCK_ADAPTIVE) return ENS_EINVAL;
    if (!(dt != 0.0) || !std::isfinite(dt) || std::isnan(t_end) || max_steps < 0) return ENS_EINVAL;
    if (!e->have_state) return ENS_ESTATE;
    ENS_ON_DEVICE(e);
    cudaStream_t s = (cudaStream_t)stream;
    ensd::StepArgs a{};
    a.dt = dt;
    a.t_end = t_end;
    a.hh = 0.5 * dt;
    a.te = dt > 0.0 ? t_end : -t_end;
    a.max_steps = max_steps;
    const double rc2 = e->r_close * e->r_close;
    double re2 = e->r_eject * e->r_eject;
    if (!(re2 < DBL_MAX)) re2 = DBL_MAX;
    memcpy(&a.rc2_bits, &rc2, 8);
    memcpy(&a.re2_bits, &re2, 8);
    {   // coordinate filter of the step loops' quick test: |x_c| < ce for all three components => |x|^2 < re2, with a
        // margin of one high-word unit (2^-20 relative) against the rounding of the exact sum
        const double ce = std::sqrt(re2 / 3.0);
        unsigned long long b;
        memcpy(&b, &ce, 8);
        a.ce_hi = (unsigned)(b >> 32);
        a.ce_hi = a.ce_hi > 0u ? a.ce_hi - 1u : 0u;  // 0: the quick test always fails (the exact logic decides)
        a.cex_hi = a.ce_hi > 0x00400000u ? a.ce_hi - 0x00100000u : 0u;  // ce / 2, ce / 4 (0: the quick test always fails)
        a.ceq_hi = a.ce_hi > 0x00400000u ? a.ce_hi - 0x00200000u : 0u;
        memcpy(&b, &e->r_close, 8);
        a.rc1_hi = (unsigned)(b >> 32) & 0x7fffffffu;
    }
    ensd::fill_step_constants(a);
    a.counter = e->counter;
    a.order = nullptr;
    a.slice_done = e->slice_done;
    a.rk_eps = e->rk_eps;
    if (integrator == ENS_HERMITE_ADAPTIVE || integrator == ENS_RKCK_ADAPTIVE) {
        CU(cudaMemsetAsync(e->counter, 0, sizeof(unsigned long long), s));
        if (!e->tune.adaptive_unordered && e->order.idx_out) {
            CU(ensd::adaptive_order(e->v, t_end, e->order, s));
            a.order = e->order.idx_out;
            e->launches += 1;  // the key kernel (the sort is cub's)
        }
    }
    const ensd::KernelInfo& ki = integrator == ENS_HERMITE            ? e->hermite
                                 : integrator == ENS_HERMITE_ADAPTIVE ? e->hermite_adaptive
                                 : integrator == ENS_HERMITE_CARRY    ? e->hermite_carry
                                 : integrator == ENS_RKCK             ? e->rkck
                                 : integrator == ENS_RKCK_ADAPTIVE    ? e->rkck_adaptive
                                 : integrator == ENS_MVS_MERGED       ? e->mvs_merged
                                                                      : e->mvs;
    if (!ki.fn) return ENS_EUNSUPPORTED;
    const int threads = e->tune.threads ? e->tune.threads : ki.threads;
    const void* fn = ki.fn;
    CU(cudaEventRecord(e->ev0, s));
    cudaError_t err = (integrator == ENS_MVS || integrator == ENS_MVS_MERGED)
                          ? ensd::launch_mvs(e->v, a, integrator == ENS_MVS_MERGED, threads, s, &e->last_blocks)
                      : (integrator == ENS_RKCK || integrator == ENS_RKCK_ADAPTIVE)
                          ? ensd::launch_rkck(e->v, a, integrator == ENS_RKCK_ADAPTIVE, threads, s, &e->last_blocks)
                          : ensd::launch_hermite(e->v, a, integrator == ENS_HERMITE_ADAPTIVE ? 1 : integrator == ENS_HERMITE_CARRY ? 2 : 0,
                                                 e->tune, s, &e->last_blocks, &fn);
    if (err != cudaSuccess) return cuda_fail(err, "ens_integrate launch");
    CU(cudaEventRecord(e->ev1, s));
    e->last_fn = fn;
    e->launches += 1;
    e->timed = true;
    return ENS_OK;
}

int ens_get_state(const ens_t* e, double* pos, double* vel, double* time, int32_t* status, int64_t* nsteps,
                  int memspace, void* stream) {
    if (!e || (memspace != ENS_HOST && memspace != ENS_DEVICE)) return ENS_EINVAL;
    if (!e->have_state) return ENS_ESTATE;
    ENS_ON_DEVICE(e);
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t n = e->v.n_sys, nb = e->v.n_body;
    const cudaMemcpyKind kind = memspace == ENS_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
    if (memspace == ENS_HOST && (pos || vel)) {
        const int rc = ensure_stage(e);
        if (rc) return rc;
    }
    const bool dev = memspace == ENS_DEVICE;
    if (pos || vel || (dev && (time || status || nsteps))) {  // one launch
        double* dp = !pos ? nullptr : dev ? pos : e->stage;
        double* dv = !vel ? nullptr : dev ? vel : e->stage + n * nb * 3;
        CU(launch_unpack(e->v, dp, dv, dev ? time : nullptr, dev ? status : nullptr, dev ? nsteps : nullptr, s));
        e->launches += 1;
        if (!dev) {
            if (pos) CU(cudaMemcpyAsync(pos, dp, sizeof(double) * n * nb * 3, kind, s));
            if (vel) CU(cudaMemcpyAsync(vel, dv, sizeof(double) * n * nb * 3, kind, s));
        }
    }
    if (!dev) {  // the per-system rows are contiguous in the SoA: straight copies
        if (time) CU(cudaMemcpyAsync(time, e->v.time, sizeof(double) * n, kind, s));
        if (status) CU(cudaMemcpyAsync(status, e->v.status, sizeof(int32_t) * n, kind, s));
        if (nsteps) CU(cudaMemcpyAsync(nsteps, e->v.nsteps, sizeof(int64_t) * n, kind, s));
    }
    CU(cudaGetLastError());
    if (memspace == ENS_HOST) CU(cudaStreamSynchronize(s));
    return ENS_OK;
}

int ens_energy(const ens_t* e, double* E, double* L, int memspace, void* stream) {
    if (!e || !E || (memspace != ENS_HOST && memspace != ENS_DEVICE)) return ENS_EINVAL;
    if (!e->have_state) return ENS_ESTATE;
    ENS_ON_DEVICE(e);
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t n = e->v.n_sys;
    double *dE = E, *dL = L;
    if (memspace == ENS_HOST) {
        const int rc = ensure_stage(e);
        if (rc) return rc;
        dE = e->stage_small;
        dL = L ? e->stage_small + n : nullptr;
    }
    switch (e->v.n_body) {
#define X(N_) \
    case N_: energy_kernel<N_><<<(unsigned)((n + 127) / 128), 128, 0, s>>>(e->v, dE, dL); break;
        ENS_FOR_EACH_NB(X)
#undef X
    }
    e->launches += 1;
    CU(cudaGetLastError());
    if (memspace == ENS_HOST) {
        CU(cudaMemcpyAsync(E, dE, sizeof(double) * n, cudaMemcpyDeviceToHost, s));
        if (L) CU(cudaMemcpyAsync(L, dL, sizeof(double) * n * 3, cudaMemcpyDeviceToHost, s));
        CU(cudaStreamSynchronize(s));
    }
    return ENS_OK;
}

int ens_log_enable(ens_t* e, int64_t capacity, void* stream) {
    if (!e || capacity < 0) return ENS_EINVAL;
    ENS_ON_DEVICE(e);
    cudaStream_t s = (cudaStream_t)stream;
    CU(cudaStreamSynchronize(s));
    LogView& g = e->log;
    cudaFree(g.cursor); cudaFree(g.last); cudaFree(g.sys); cudaFree(g.nsteps);
    cudaFree(g.time); cudaFree(g.status); cudaFree(g.pos); cudaFree(g.vel);
    g = LogView{};
    if (capacity == 0) return ENS_OK;
    const int64_t n3 = (int64_t)e->v.n_body * 3;
    CU(cudaMalloc(&g.cursor, sizeof(unsigned long long)));
    CU(cudaMalloc(&g.last, sizeof(int64_t) * e->v.n_pad));
    CU(cudaMalloc(&g.sys, sizeof(int64_t) * capacity));
    CU(cudaMalloc(&g.nsteps, sizeof(int64_t) * capacity));
    CU(cudaMalloc(&g.time, sizeof(double) * capacity));
    CU(cudaMalloc(&g.status, sizeof(int32_t) * capacity));
    CU(cudaMalloc(&g.pos, sizeof(double) * capacity * n3));
    CU(cudaMalloc(&g.vel, sizeof(double) * capacity * n3));
    g.capacity = capacity;
    log_reset_kernel<<<(unsigned)((e->v.n_pad + 255) / 256), 256, 0, s>>>(g.last, e->v.n_pad, g.cursor);
    e->launches += 1;
    CU(cudaGetLastError());
    return ENS_OK;
}

int ens_integrate_logged(ens_t* e, int integrator, double dt, double t_end, int64_t max_steps, int64_t log_every,
                         int what, void* stream) {
    if (!e || log_every < 1 || !(what & (ENS_LOG_SNAPSHOTS | ENS_LOG_STOPS))) return ENS_EINVAL;
    // every segment is two launches enqueued from the host, whether or not systems are still running: a step budget
    // that is really "until t_end" must come with a log_every that keeps the segment count sane
    if (max_steps / log_every > 1000000) return ENS_EINVAL;
    if (e->log.capacity == 0) return ENS_ESTATE;
    ENS_ON_DEVICE(e);
    cudaStream_t s = (cudaStream_t)stream;
    int64_t done = 0;
    do {  // segments of log_every steps, each followed by the log kernel: all enqueued, no host round trip
        const int64_t seg = (max_steps - done < log_every) ? (max_steps - done) : log_every;
        const int rc = ens_integrate(e, integrator, dt, t_end, seg, stream);
        if (rc != ENS_OK) return rc;
        log_kernel<<<(unsigned)((e->v.n_sys + 127) / 128), 128, 0, s>>>(e->v, e->log, what);
        e->launches += 1;
        CU(cudaGetLastError());
        done += seg;
    } while (done < max_steps);
    return ENS_OK;
}

int ens_log_read(const ens_t* e, int64_t* n_records, int64_t* n_dropped, int64_t* sys, int64_t* nsteps, double* time,
                 int32_t* status, double* pos, double* vel, int64_t max_records, int memspace, void* stream) {
    if (!e || !n_records || max_records < 0 || (memspace != ENS_HOST && memspace != ENS_DEVICE)) return ENS_EINVAL;
    if (e->log.capacity == 0) return ENS_ESTATE;
    ENS_ON_DEVICE(e);
    cudaStream_t s = (cudaStream_t)stream;
    const LogView& g = e->log;
    unsigned long long cur = 0;
    CU(cudaMemcpyAsync(&cur, g.cursor, sizeof cur, cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));  // the record count is a host value: this call always waits for the stream
    const int64_t stored = (int64_t)cur < g.capacity ? (int64_t)cur : g.capacity;
    const int64_t n = stored < max_records ? stored : max_records;
    *n_records = n;
    if (n_dropped) *n_dropped = (int64_t)cur - stored;
    const cudaMemcpyKind kind = memspace == ENS_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
    const int64_t n3 = (int64_t)e->v.n_body * 3;
    if (n > 0) {
        if (sys) CU(cudaMemcpyAsync(sys, g.sys, sizeof(int64_t) * n, kind, s));
        if (nsteps) CU(cudaMemcpyAsync(nsteps, g.nsteps, sizeof(int64_t) * n, kind, s));
        if (time) CU(cudaMemcpyAsync(time, g.time, sizeof(double) * n, kind, s));
        if (status) CU(cudaMemcpyAsync(status, g.status, sizeof(int32_t) * n, kind, s));
        if (pos) CU(cudaMemcpyAsync(pos, g.pos, sizeof(double) * n * n3, kind, s));
        if (vel) CU(cudaMemcpyAsync(vel, g.vel, sizeof(double) * n * n3, kind, s));
        if (memspace == ENS_HOST) CU(cudaStreamSynchronize(s));
    }
    return ENS_OK;
}

int ens_get_info(const ens_t* e, int64_t out[10]) {
    if (!e || !out) return ENS_EINVAL;
    ENS_ON_DEVICE(e);
    const ensd::KernelInfo* all[] = {&e->mvs, &e->hermite_adaptive, &e->hermite_carry, &e->hermite_sliced, &e->rkck,
                                     &e->rkck_adaptive, &e->mvs_merged};
    const ensd::KernelInfo* ki = &e->hermite;
    for (const ensd::KernelInfo* c : all)
        if (e->last_fn && e->last_fn == c->fn) ki = c;
    const int threads = e->tune.threads ? e->tune.threads : ki->threads;
    out[0] = e->v.n_pad;
    out[1] = ki->shape.L;
    out[2] = ki->shape.B;
    out[3] = threads;
    const int64_t sys_per_warp = 32 / (ki->shape.L > 0 ? ki->shape.L : 1);
    const int64_t warps = (e->v.n_sys + sys_per_warp - 1) / sys_per_warp;
    out[4] = e->last_blocks ? e->last_blocks : (warps + threads / 32 - 1) / (threads / 32);
    out[5] = out[6] = out[8] = 0;
    out[9] = ki->fn == e->hermite_sliced.fn && ki->fn ? 1 : 0;
    if (ki->fn) {
        cudaFuncAttributes fa;
        CU(cudaFuncGetAttributes(&fa, ki->fn));
        out[5] = fa.numRegs;
        out[8] = (int64_t)fa.localSizeBytes;
        int nb = 0;
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, ki->fn, threads, (size_t)(threads / 32) * ki->smem_bytes_per_warp));
        out[6] = nb;
    }
    out[7] = e->launches;
    return ENS_OK;
}

int ens_last_kernel_ms(const ens_t* e, float* ms) {
    if (!e || !ms) return ENS_EINVAL;
    if (!e->timed) return ENS_ESTATE;
    ENS_ON_DEVICE(e);
    CU(cudaEventSynchronize(e->ev1));
    CU(cudaEventElapsedTime(ms, e->ev0, e->ev1));
    return ENS_OK;
}

int ens_fp64_peak(int64_t iters, double* lane_fma_per_s, void* stream) {
    if (iters < 1 || !lane_fma_per_s) return ENS_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    struct Scratch {  // released on every return path
        double* out = nullptr;
        cudaEvent_t a = nullptr, b = nullptr;
        ~Scratch() {
            if (a) cudaEventDestroy(a);
            if (b) cudaEventDestroy(b);
            cudaFree(out);
        }
    } w;
    CU(cudaMalloc(&w.out, sizeof(double)));
    CU(cudaEventCreate(&w.a));
    CU(cudaEventCreate(&w.b));
    const int blocks = sms * 8, threads = 256;  // 64 warps per SM
    dfma_kernel<<<blocks, threads, 0, s>>>(iters / 8 + 1, 1.0, w.out);  // warm-up
    CU(cudaEventRecord(w.a, s));
    dfma_kernel<<<blocks, threads, 0, s>>>(iters, 1.0, w.out);
    CU(cudaEventRecord(w.b, s));
    CU(cudaEventSynchronize(w.b));
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, w.a, w.b));
    CU(cudaGetLastError());
    *lane_fma_per_s = (double)blocks * threads * (double)iters * 64.0 / (ms * 1e-3);
    return ENS_OK;
}

int ens_test_set_option(ens_t* e, int option, int64_t value) {
    if (!e || value < 0) return ENS_EINVAL;
    switch (option) {
        case ENS_OPT_THREADS:
            if (value != 0 && (value < 32 || value > 1024 || (value & 31))) return ENS_EINVAL;
            e->tune.threads = (int)value;
            return ENS_OK;
        case ENS_OPT_ADAPTIVE_UNORDERED: e->tune.adaptive_unordered = value != 0; return ENS_OK;
        case ENS_OPT_SLICE_MODE:
            if (value > 2) return ENS_EINVAL;
            e->tune.slice_mode = (int)value;
            return ENS_OK;
        case ENS_OPT_SLICE_STEPS: e->tune.slice_steps = value; return ENS_OK;
        case ENS_OPT_SLICE_WARPS_PER_SM:
            if (value > 64) return ENS_EINVAL;
            e->tune.slice_warps_per_sm = (int)value;
            return ENS_OK;
    }
    return ENS_EINVAL;
}

}  // extern "C"
