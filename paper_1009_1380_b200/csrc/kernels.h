// kernels.h -- device-side view of a plan and the kernel launchers (internal).
#pragma once
#include <cuda_runtime.h>

#include "radon_internal.h"

namespace radon {

struct DevicePlan {
    int N = 0, G = 0, n_angles = 0, n_det = 0, LP = 0;   // LP: FFT length of the projection DFT
    // tables
    double2 *cs = nullptr;        // per angle (G/n)(cos, sin), fp64
    float *lut = nullptr;         // LUT_S x LUT_ROW (only with RADON_KB_LUT)
    KbPoly kb;                    // polynomial pieces of the Kaiser-Bessel kernel
    float *deapod = nullptr;      // N
    float2 *tw_G = nullptr;       // twiddles for length G
    float2 *tw_P = nullptr;       // twiddles for length LP
    float2 *chirp_a = nullptr, *chirp_b = nullptr, *chirp_hf = nullptr;   // hf == nullptr: direct FFT
    // schedules
    GatherCta *gather_ctas = nullptr;   int n_gather_ctas = 0;
    Slot *gather_slots = nullptr;
    ScatterCta *scatter_ctas = nullptr; int n_scatter_ctas = 0;
    Slot *scatter_slots = nullptr;
    MergeJob *merge_jobs = nullptr;     int n_merge_jobs = 0;
    float2 *scratch = nullptr;          // partial rectangles of split tiles
};

bool fft_length_supported(int L);
int init_kernel_attributes();
long long launch_count();

// F3 / A2 (+ merge)
int launch_gather(const DevicePlan &p, const float2 *grid, float2 *polar, cudaStream_t st);
int launch_scatter(const DevicePlan &p, const float2 *polar, float2 *grid, cudaStream_t st);
// which: 0 colpass_fwd (x -> T), 1 rowpass_fwd (T -> grid), 2 rowpass_inv (grid -> T), 3 colpass_inv (T -> x)
int launch_fft2d_pass(int which, const DevicePlan &p, const void *in, void *out, cudaStream_t st);
// inv == false: sinogram -> polar (A1); inv == true: polar -> sinogram (F4)
int launch_proj(bool inv, const DevicePlan &p, const float *in, float *out, cudaStream_t st);

}  // namespace radon
