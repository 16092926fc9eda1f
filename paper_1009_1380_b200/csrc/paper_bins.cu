// paper_bins.cu -- the paper's own GPU design for the gridding step, as a measured comparison
// (prior art, not the product path: radon_grid_only / radon_adjoint use the
// plan-time round schedules of gridding.cu).
//
// "we partition the regular and irregular samples into bins such that the amount of
// computation is approximately constant.  The load balancing algorithm starts by considering one
// bin containing all the points, and recursively divides the most computationally intensive bin
// into four equally sized bins ...  We then launch one thread block per bin.  When the number of
// samples does not fit in shared memory we assign all threads to each grid point and use
// coalesced memory reads to evaluate the contribution of each sample to the grid point.  When it
// does fit in shared memory we assign one thread per grid point and loop through all the samples
// (in shared memory) to evaluate their contribution to each grid point."
//
// Bins come from build_paper_bins (plan_host.cpp).  Both strategies are output driven: a grid
// point gathers K(x_i - x_r, y_i - y_r) G(x_i, y_i) from the bin's samples (D == 1)
// with the same tap rule and the same Kaiser-Bessel weights as the product kernels, so the
// result differs from radon_grid_only only by the order of the additions.
#include "kernels.h"
#include "taps.cuh"

namespace radon {

constexpr int PB_THREADS = 256;
constexpr int PB_STAGE = 1024;                  // samples that "fit in shared memory" (64 bytes each)
template <int KW>
struct __align__(16) StagedSample {
    float wx[KW], wy[KW];                       // tap weights along x and y
    float vr, vi;                               // sample value
    int bx, by;                                 // base cell of the footprint (may lie outside [0, G))
};
static_assert(sizeof(StagedSample<6>) == 64 && sizeof(StagedSample<8>) == 80 && sizeof(StagedSample<4>) == 48, "staged sample layout");

template <int KW>
__device__ __forceinline__ void stage_sample(const PaperBinEntry en, const float2 *__restrict__ polar,
                                             const double2 *__restrict__ cs, const KbPoly &kp, int G, int n_det,
                                             StagedSample<KW> &s)
{
    const int a = (int)(en.ak >> 16), k = (int)(en.ak & 0xffff);
    const double2 d = __ldg(&cs[a]);
    const double halfG = 0.5 * (double)G, jj = (double)(k - n_det / 2);
    Taps<KW> tp;
    sample_taps_dir<KW>(d, kp, k, n_det / 2, halfG, tp);
#pragma unroll
    for (int l = 0; l < KW; ++l) { s.wx[l] = tp.wx[l]; s.wy[l] = tp.wy[l]; }
    const float2 v = __ldg(&polar[(size_t)a * n_det + k]);
    s.vr = v.x; s.vi = v.y;
    s.bx = (int)ceil(fma(jj, d.x, halfG) - 0.5 * KW) + ((en.shift & 3) - 1) * G;
    s.by = (int)ceil(fma(jj, d.y, halfG) - 0.5 * KW) + (((en.shift >> 2) & 3) - 1) * G;
}

// one thread block per bin
template <int KW>
__global__ void __launch_bounds__(PB_THREADS)
paper_bins_kernel(const float2 *__restrict__ polar, float2 *__restrict__ grid, const PaperBin *__restrict__ bins,
                  const PaperBinEntry *__restrict__ entries, const double2 *__restrict__ cs, const KbPoly kp,
                  int G, int n_det)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    StagedSample<KW> *st = reinterpret_cast<StagedSample<KW> *>(smem_raw);
    __shared__ float2 red[PB_THREADS / 32];
    const PaperBin bin = bins[blockIdx.x];
    const PaperBinEntry *list = entries + bin.first;
    const int n_cells = bin.w * bin.h;

    if (bin.count <= PB_STAGE) {
        // "it does fit in shared memory": one thread per grid point, loop through the staged samples
        for (int i = threadIdx.x; i < bin.count; i += PB_THREADS) stage_sample<KW>(list[i], polar, cs, kp, G, n_det, st[i]);
        __syncthreads();
        for (int c = threadIdx.x; c < n_cells; c += PB_THREADS) {
            const int X = bin.x0 + c % bin.w, Y = bin.y0 + c / bin.w;
            float ar = 0.f, ai = 0.f;
            for (int i = 0; i < bin.count; ++i) {
                const unsigned lx = (unsigned)(X - st[i].bx), ly = (unsigned)(Y - st[i].by);
                if (lx < (unsigned)KW && ly < (unsigned)KW) {
                    const float w = st[i].wx[lx] * st[i].wy[ly];
                    ar = fmaf(st[i].vr, w, ar);
                    ai = fmaf(st[i].vi, w, ai);
                }
            }
            grid[(size_t)Y * G + X] = make_float2(ar, ai);
        }
        return;
    }
    // "the number of samples does not fit in shared memory": all threads on each grid point,
    // coalesced reads of the sample list, block reduction (fixed order)
    for (int c = 0; c < n_cells; ++c) {
        const int X = bin.x0 + c % bin.w, Y = bin.y0 + c / bin.w;
        float ar = 0.f, ai = 0.f;
        for (int i = threadIdx.x; i < bin.count; i += PB_THREADS) {
            StagedSample<KW> s;
            const PaperBinEntry en = list[i];
            // cheap reject before the weights: base cell from the fp64 coordinates
            const int a = (int)(en.ak >> 16), k = (int)(en.ak & 0xffff);
            const double2 d = __ldg(&cs[a]);
            const double halfG = 0.5 * (double)G, jj = (double)(k - n_det / 2);
            const int bx = (int)ceil(fma(jj, d.x, halfG) - 0.5 * KW) + ((en.shift & 3) - 1) * G;
            const int by = (int)ceil(fma(jj, d.y, halfG) - 0.5 * KW) + (((en.shift >> 2) & 3) - 1) * G;
            const unsigned lx = (unsigned)(X - bx), ly = (unsigned)(Y - by);
            if (lx < (unsigned)KW && ly < (unsigned)KW) {
                stage_sample<KW>(en, polar, cs, kp, G, n_det, s);
                float wx = 0.f, wy = 0.f;
#pragma unroll
                for (int l = 0; l < KW; ++l) { wx = (l == (int)lx) ? s.wx[l] : wx; wy = (l == (int)ly) ? s.wy[l] : wy; }
                ar = fmaf(s.vr, wx * wy, ar);
                ai = fmaf(s.vi, wx * wy, ai);
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            ar += __shfl_xor_sync(0xffffffffu, ar, o);
            ai += __shfl_xor_sync(0xffffffffu, ai, o);
        }
        __syncthreads();
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = make_float2(ar, ai);
        __syncthreads();
        if (threadIdx.x == 0) {
            float sr = 0.f, si = 0.f;
            for (int w = 0; w < PB_THREADS / 32; ++w) { sr += red[w].x; si += red[w].y; }
            grid[(size_t)Y * G + X] = make_float2(sr, si);
        }
    }
}

int launch_paper_bins(const DevicePlan &p, const PaperBin *bins, int n_bins, const PaperBinEntry *entries,
                      const float2 *polar, float2 *grid, cudaStream_t st)
{
    RADON_FOR_W(p.W, {
        const size_t smem = (size_t)PB_STAGE * sizeof(StagedSample<WW>);
        if (set_smem(paper_bins_kernel<WW>, smem)) return -1;
        launch_pdl(false, paper_bins_kernel<WW>, n_bins, PB_THREADS, smem, st, polar, grid, bins, entries, p.cs, p.kb, p.G, p.n_det);
    })
    count_launch();
    return 0;
}

}  // namespace radon
