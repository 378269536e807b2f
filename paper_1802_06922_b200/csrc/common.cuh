// Internal header of libqmcb200: handle layouts, error plumbing, small device helpers.
// Not part of the public boundary (that is include/qmc_b200.h).
#pragma once
#include <cuda_runtime.h>
#include <stdarg.h>
#include <stdint.h>
#include <stdio.h>

#include <vector>

#include "qmc_b200.h"

namespace qmc {

constexpr int kWarp = 32;
constexpr int kMaxNel = 2048;       // rows are held in registers: 64 doubles per lane at most
constexpr int kSpoBatch = 16;       // electron steps per SPO-VGL launch in rank-1 mode (delayed: the window)

void set_error(const char *fmt, ...);
void count_launch(int n = 1);

#define QMC_CUDA(call)                                                                     \
    do {                                                                                   \
        cudaError_t e__ = (call);                                                          \
        if (e__ != cudaSuccess) {                                                          \
            qmc::set_error("%s:%d: %s -> %s", __FILE__, __LINE__, #call,                   \
                           cudaGetErrorString(e__));                                       \
            return QMC_ECUDA;                                                              \
        }                                                                                  \
    } while (0)

// Same, running `cleanup` before the error return.
#define QMC_CUDA_OR(call, cleanup)                                                         \
    do {                                                                                   \
        cudaError_t e__ = (call);                                                          \
        if (e__ != cudaSuccess) {                                                          \
            qmc::set_error("%s:%d: %s -> %s", __FILE__, __LINE__, #call,                   \
                           cudaGetErrorString(e__));                                       \
            cleanup;                                                                       \
            return QMC_ECUDA;                                                              \
        }                                                                                  \
    } while (0)

#define QMC_REQUIRE(cond, ...)                                                             \
    do {                                                                                   \
        if (!(cond)) {                                                                     \
            qmc::set_error(__VA_ARGS__);                                                   \
            return QMC_EINVAL;                                                             \
        }                                                                                  \
    } while (0)

// Launch check: catches bad configurations at once (no synchronisation).
#define QMC_LAUNCHED()                                                                     \
    do {                                                                                   \
        qmc::count_launch();                                                               \
        QMC_CUDA(cudaGetLastError());                                                      \
    } while (0)

// What the SPO kernels need to know about the table (passed by value).
struct SplineView {
    const float *coefs;   // [nx][ny][nz][np]
    int nx, ny, nz, norb, np;
    double linv[9];       // lattice^-1, row-major: u_d = sum_j r_j linv[3j+d]
    double jac[9];        // jac[3j+d] = linv[3j+d] * N_d = d s_d / d r_j
    double metric[6];     // G_de = sum_j jac[j][d] jac[j][e]: xx,yy,zz,xy,xz,yz
    int half_twist[3];    // 1: twist angle pi along cell vector d (eq. 43, R:A23); 0: periodic
};

}  // namespace qmc

struct qmc_spline {
    qmc::SplineView view;
    float *coefs;         // owned
    size_t bytes;
};

struct qmc_det {
    const qmc_spline *spline;   // not owned; shape checks and det_init only
    int nw, nel, ld, delay;
    int device, nsm;            // the CUDA device the handle lives on and its SM count (grid sizing)
    int np;                     // spline row pitch (floats)
    double *B;                  // [nw][nel][ld]   (A^-1)^T, pad columns zero (fp64 storage; NULL when b32)
    int b32;                    // 1: the inverse is STORED in fp32 (R:A19): Bf is used instead of B
    float *Bf;                  // [nw][nel][ld]   the same matrix in fp32 (NULL unless b32)
    double *logdet;             // [nw]
    int *sign;                  // [nw]
    long long *naccept;         // [nw]
    // scratch owned by the handle
    int spo_batch;              // electron steps whose SPO-VGL is evaluated per launch (qmc_sweep)
    float *vgl;                 // [spo_batch][nw][5][np]   v, gx, gy, gz, lap of the proposals of a batch
    // delayed mode: the SPO-VGL of window i+1 is evaluated on a second stream while window i is
    // flushed (the proposals of a window depend on nothing the previous window changes)
    float *vgl_buf[2];          // vgl_buf[0] == the allocation vgl points into first; [1] only when overlap is on
    cudaStream_t aux;           // second stream (non-blocking), created on first use
    cudaEvent_t ev_spo[2], ev_main;
    int overlap;                // 1: overlap enabled (delay >= 2 and QMC_SWEEP_OVERLAP != 0)
    // drift moves (qmc_sweep_ex drift_tau > 0): allocated on first use
    float *vgl_cur;             // [kSpoBatch][nw][5][np] SPO-VGL at the CURRENT positions of a batch of electrons
    double *rprop, *fcur, *tfac;   // [nw][3], [nw][3], [nw]: proposal, F_k(r), T(r'->r)/T(r->r') of the current step
    double *jas_dj;             // [max(delay, 1)][nw] Jastrow dJ of the steps of a window / exp(-2 dJ) of a step (on first use)
    double *rowk;               // [nw][ld]      copy of row iel of B taken before the update
    double *ratio;              // [nw]      ratio of the current step (ratio_rowcopy_kernel -> sm_update_kernel)
    unsigned char *acc;         // [nw]
    // delayed-update window (delay >= 2)
    int *win_count;             // [nw]           accepted rows pending
    int *win_iel;               // [nw][delay]    their electron indices
    int *win_slot;              // [nw][delay]    slot of row / vector l in win_rows / win_vec
    float *win_phi;             // [nw][delay][np] orbital vectors appended by qmc_det_accept_update
    double *win_rows;           // [nw][delay][ld] rows B0[k_l] (qmc_det_accept_update), turned into R' = S^-T Rows for the flush
    int win_rows_raw;           // win_rows still holds the raw rows (the flush converts them first)
    const float *win_vec;       // where the flush finds the vectors: win_phi, or the SPO-VGL scratch (qmc_sweep)
    size_t win_vec_wstride, win_vec_sstride;   // its walker and slot strides (floats)
    double *win_sinv;           // [nw][delay][delay] inverse of S
    int *win_full;              // [1] set when any walker's window is full
    int accept_windows;         // QMC_DET_ACCEPT_WINDOWS: windows close on delay accepted moves; spo_batch = steps per window
    int *cur;                   // [2][nw] accept_windows: electron cursor of every walker within the current sweep, and
                                //   (second half, `ev`) the electron up to which its proposals' SPO-VGL has been evaluated
    int vgl_ring;               // accept_windows: the SPO-VGL scratch is a ring of this many slots (2 x spo_batch),
                                //   slot = electron % ring: proposals a window did not reach are reused by the next
    int win_kend;               // end of the electron range of the sweep in progress (accept_windows)
    int host_pending;           // electron steps appended to the open window (host bookkeeping)
    unsigned char *win_host_iel;   // host [nel]: electrons touched in the open window
    double *kin_lap;            // [nw][nel] scratch of qmc_det_kinetic (allocated on first use)
    // device staging of qmc_sweep_host (grown on demand)
    void *stage;
    size_t stage_bytes;
    // per-kernel timing (qmc_det_profile): CUDA events around every launch of a sweep
    int prof_on;
    std::vector<cudaEvent_t> *prof_events;   // pool, pairs (start, stop)
    std::vector<int> *prof_kinds;            // kind of pair i
    size_t prof_used;                        // events handed out since the last reset
};

// Run `...` with TB = the handle's storage type and Bp = its matrix.
#define QMC_WITH_B(d, TB, Bp, ...)                                                         \
    do {                                                                                   \
        if ((d)->b32) { using TB = float; TB *Bp = (d)->Bf; (void)Bp; __VA_ARGS__; }       \
        else { using TB = double; TB *Bp = (d)->B; (void)Bp; __VA_ARGS__; }                \
    } while (0)

namespace qmc {
enum ProfKind { kProfSpoRatio = 0, kProfUpdate = 1, kProfDelayedRatio = 2, kProfDelayedAccept = 3,
                kProfDelayedFlush = 4, kProfRatio = 5, kProfKinds = 6 };
static_assert(kProfKinds == QMC_PROF_KINDS, "qmc_b200.h and common.cuh disagree on the profiling kinds");
// Record a start / stop event pair around a launch when profiling is enabled (no-ops otherwise).
void prof_start(qmc_det *d, int kind, cudaStream_t s);
void prof_stop(qmc_det *d, cudaStream_t s);
}

namespace qmc {

__device__ __forceinline__ double warp_sum(double x)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

// Deterministic block sum (fixed order); result valid in every thread.  `red` holds >= 33 doubles.
__device__ __forceinline__ double block_sum(double x, double *red)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
    x = warp_sum(x);
    __syncthreads();
    if (lane == 0) red[wid] = x;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int i = 0; i < nwarp; ++i) s += red[i];
        red[32] = s;
    }
    __syncthreads();
    return red[32];
}

// Storage type of the inverse (double, or float for the single-precision inverse of PAPER.md L82,
// R:A19): two consecutive elements as fp64, and back (one rounding to nearest even when TB = float).
__device__ __forceinline__ double2 ld2(const double *p) { return *reinterpret_cast<const double2 *>(p); }
__device__ __forceinline__ double2 ld2(const float *p)
{
    const float2 f = *reinterpret_cast<const float2 *>(p);
    return make_double2((double)f.x, (double)f.y);
}
__device__ __forceinline__ void st2(double *p, double2 v) { *reinterpret_cast<double2 *>(p) = v; }
__device__ __forceinline__ void st2(float *p, double2 v) { *reinterpret_cast<float2 *>(p) = make_float2((float)v.x, (float)v.y); }

__device__ __forceinline__ float4 ldg_stream(const float4 *p)
{
    float4 r;
    asm("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w)
                 : "l"(p));
    return r;
}

}  // namespace qmc
