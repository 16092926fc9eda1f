// kernels.h -- device-side view of a plan and the kernel launchers (internal).
#pragma once
#include <mutex>
#include <set>
#include <utility>
#include <cuda_runtime.h>

#include "radon_internal.h"

namespace radon {

struct DevicePlan {
    int N = 0, G = 0, n_angles = 0, n_det = 0, LP = 0;   // LP: FFT length of the projection DFT
    int W = 6;                    // Kaiser-Bessel width (4, 6 or 8)
    int st_y = ST_Y;              // rows of a scatter tile (Geometry::st_y)
    int n_sm = 148;               // multiprocessors of the device (persistent grids)
    bool pdl = false;             // programmatic dependent launch between the kernels of a call
    // tables
    double2 *cs = nullptr;        // per angle (G/n)(cos, sin), fp64
    KbPoly kb;                    // polynomial pieces of the Kaiser-Bessel kernel
    float *deapod = nullptr;      // N
    float2 *tw_G = nullptr;       // twiddles for length G
    float2 *tw_sub = nullptr;     // G = 3 or 5 times a power of two P: twiddles for length P (fft2d_composite.cu)
    float2 *tw_P = nullptr;       // twiddles for length LP
    float2 *chirp_a = nullptr, *chirp_b = nullptr, *chirp_hf = nullptr;   // hf == nullptr: direct FFT
    // schedules: [0] every sample / whole grid (arbitrary complex data: the test hooks),
    //            [1] Hermitian half (real image / real sinogram: radon_forward, radon_adjoint)
    struct Sched {
        GatherCta *gather_ctas = nullptr;   int n_gather_ctas = 0;      // work items
        int *gather_worker_begin = nullptr; int n_gather_workers = 0;   // persistent CTAs
        Slot *gather_slots = nullptr;
        ScatterCta *scatter_ctas = nullptr; int n_scatter_ctas = 0;
        Slot *scatter_slots = nullptr;
        MergeJob *merge_jobs = nullptr;     int n_merge_jobs = 0;
        int dc_jobs[MAX_DC_JOBS] = {0, 0, 0, 0}; int n_dc_jobs = 0;    // merge jobs that add the j = 0 sum
    } sched[2];
};

// A4 epilogue of a solver iteration: x <- S_tau(x - alpha * g) in place, g the freshly computed adjoint
struct IstaUpdate { float alpha = 0.f, tau = 0.f; };

bool fft_length_supported(int L);            // power of two in [16, 8192], or 3 / 5 times a power of two in [16, 2048]
bool fft_composite_split(int L, int *P_out, int *PR_out);
int launch_fft2d_composite(int which, const DevicePlan &p, const void *in, void *out, int flag, cudaStream_t st,
                           const IstaUpdate *upd);
int init_kernel_attributes();
long long launch_count();
void count_launch(long long n = 1);

// Opt a kernel in to more than 48 KB of dynamic shared memory: once per (device, kernel); the
// attribute call costs microseconds of host time, which a batch of back-to-back launches feels.
template <typename F>
static inline int set_smem(F kernel, size_t bytes)
{
    if (bytes <= 40 * 1024) return 0;        // static shared memory counts towards the 48 KB default too
    static std::mutex mu;
    static std::set<std::pair<int, const void *>> done;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1;
    const std::pair<int, const void *> key(dev, reinterpret_cast<const void *>(kernel));
    std::lock_guard<std::mutex> lock(mu);
    if (done.count(key)) return 0;
    if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess)
        return -1;
    done.insert(key);
    return 0;
}

// Programmatic dependent launch: every kernel of a call sequence is launched with the
// programmatic-stream-serialisation attribute and starts with pdl_prologue(): it waits until its
// predecessor has completed and its writes are visible; nothing touches global memory before that
// wait, so the order of the sequence is what stream order would give.  A kernel calls
// pdl_trigger() when its main work is done: once all its CTAs have, the successor's CTAs are
// scheduled onto the multiprocessors the tail of this grid leaves idle and run their set-up.
// Measured on a B200: config 1 pair 57 -> 43 us, config 2 82 -> 64 us, the paper's 180 x 1024 shape
// 71 -> 54 us; at config 4 (G = 4096), with the trigger late in every kernel, one slice at a time
// 222-230 -> 214 us, bare gridding 83.8 -> 81.9 us, bare interpolation 42.0 -> 40.8 us, the 32-slice batch
// unchanged.  RADON_PDL=0 in the environment launches plainly (A/B).
bool pdl_enabled();                  // RADON_PDL != 0 and no graph capture of the library in progress
void pdl_suppress(bool on);          // the solver's graph capture launches plainly (measured: graph + PDL is slower)
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_prologue() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
// called where a CTA has its main work behind it (before its output phase): once every CTA of the
// grid has passed this point (or exited) the successor's CTAs may be scheduled
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
template <typename... KArgs, typename... Args>
static inline cudaError_t launch_pdl(bool pdl, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args &&...args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = (pdl && pdl_enabled()) ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}
#endif

// Dispatch a runtime power-of-two FFT length to a template instance (LL).
#define RADON_FOR_L(L, BODY)                         \
    switch (L) {                                     \
    case 16: { constexpr int LL = 16; BODY } break;  \
    case 32: { constexpr int LL = 32; BODY } break;  \
    case 64: { constexpr int LL = 64; BODY } break;  \
    case 128: { constexpr int LL = 128; BODY } break;    \
    case 256: { constexpr int LL = 256; BODY } break;    \
    case 512: { constexpr int LL = 512; BODY } break;    \
    case 1024: { constexpr int LL = 1024; BODY } break;  \
    case 2048: { constexpr int LL = 2048; BODY } break;  \
    case 4096: { constexpr int LL = 4096; BODY } break;  \
    case 8192: { constexpr int LL = 8192; BODY } break;  \
    default: return -1;                              \
    }

// F3 / A2 (+ merge)
// half: use the Hermitian-half schedule (sched[1]).  Gather: only k >= n/2 of every polar row
// is written (plus k = 0 for even n, from the ghost sample); scatter: only grid rows
// [G/2, G) and row 0 are written.
int launch_gather(const DevicePlan &p, bool half, const float2 *grid, float2 *polar, cudaStream_t st);
// scratch: room for the partial rectangles of the schedule's split tiles (one set per stream in flight)
// dcbuf: (W+1)^2 float2 per stream in flight (the summed j = 0 samples on the centre window)
// tickets: MERGE_COUNTERS zero-initialised ints per merge job per stream in flight (re-armed by the kernel)
constexpr int MERGE_COUNTERS_PER_JOB = 4;
int launch_scatter(const DevicePlan &p, bool half, const float2 *polar, float2 *grid, float2 *scratch,
                   float2 *dcbuf, int *tickets, cudaStream_t st);
// which: 0 colpass_fwd (x -> T), 1 rowpass_fwd (T -> grid; flag 1: also write every mirrored row,
// flag 2: only the mirrored rows the half gather reads, |ky| <= W/2 and |ky - G/2| <= W/2),
// 2 rowpass_inv (grid -> T; flag: fold the mirrored rows in), 3 colpass_inv (T -> x).
// T holds the rows ky = 0..G/2 only (Hermitian half), N complex each.
int launch_fft2d_pass(int which, const DevicePlan &p, const void *in, void *out, int flag, cudaStream_t st,
                      const IstaUpdate *upd = nullptr);
// inv == false: sinogram -> polar (A1); inv == true: polar -> sinogram (F4).  half (F4 only):
// the polar rows hold k >= n/2 (and k = 0 for even n); the rest is their conjugate mirror.
// dens (A1 only, may be null): per-sample density weights multiplied into the output (radon_inverse).
// sub (F4 only, may be null): a sinogram subtracted from the result (the residual Radon{x} - data);
// q (may be null): basis of the polynomial sinogram filter (n_det x FILTER_MAXQ, orders <= 3), applied
// along every projection to the output (F4, after `sub`) or to the input (A1): PAPER.md:27, :31.
struct ProjExtra { const float *sub = nullptr; const float *q = nullptr; };
int launch_proj(bool inv, bool half, const DevicePlan &p, const float *in, float *out, const float *dens, cudaStream_t st,
                const ProjExtra &ex = ProjExtra());
// axis 0: along the detector coordinate of every projection; 1: along the angles of every detector bin
// order > 3: the basis has more than four columns
int launch_filter(const DevicePlan &p, int axis, const float *q, int order, const float *in, float *out, cudaStream_t st);


// The paper's own design, comparison only: one thread block per load-balanced bin
int launch_paper_bins(const DevicePlan &p, const PaperBin *bins, int n_bins, const PaperBinEntry *entries,
                      const float2 *polar, float2 *grid, cudaStream_t st);

}  // namespace radon
