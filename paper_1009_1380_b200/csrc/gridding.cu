// gridding.cu -- the gridding / inverse-gridding kernels of the NUFFT-Radon hot path (sm_100a).
//
//   gather_kernel    F3  inverse gridding, PAPER.md:87 (regular grid -> polar samples)
//   scatter_kernel   A2  gridding, PAPER.md:85 with D == 1 (polar samples -> regular grid)
//   merge_kernel         fixed-order sum of the partial rectangles of split tiles
//   colpass/rowpass  F1+F2 / A3+A4  de-apodise + zero-pad + 2-D FFT, and the transposed chain
//   proj kernels     F4 / A1  centred 1-D DFTs along the projections (Bluestein for any n_det)
#include "kernels.h"

#include <atomic>

namespace radon {

static std::atomic<long long> g_launches{0};
long long launch_count() { return g_launches.load(); }
void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

// =====================================================================================
// Sample coordinates and Kaiser-Bessel weights (shared by gather and scatter so that the
// two kernels use bit-identical tap positions and weights: exact transposes)
// =====================================================================================
struct Taps {
    float wx[KW], wy[KW];
};

// LUT row `it` holds, for tap l = 0..KW-1, (phi(it/S - W/2 + l), slope to the next row).
__device__ __forceinline__ void lut_weights(const float *lut, float delta, float (&w)[KW])
{
    const float t = delta * (float)LUT_S;
    int it = (int)t;
    it = min(it, LUT_S - 1);
    const float e = t - (float)it;
    const float4 *row = reinterpret_cast<const float4 *>(lut + it * LUT_ROW);
#pragma unroll
    for (int q = 0; q < KW / 2; ++q) {
        const float4 r = row[q];
        w[2 * q] = fmaf(e, r.y, r.x);
        w[2 * q + 1] = fmaf(e, r.w, r.z);
    }
}

// Polar sample (a,k) -> fractional offsets of its first tap: delta = x0 - (gx - W/2) in [0,1).
// fp64 on purpose (an fp32 product G*j/n*cos loses 2.6e-5 at G = 4096).
__device__ __forceinline__ void sample_taps(const double2 *__restrict__ cs, const float *lut, const KbPoly &kp,
                                            int a, int k, int cd, double halfG, Taps &tp)
{
    const double2 d = __ldg(&cs[a]);
    const double jj = (double)(k - cd);
    const double gx = fma(jj, d.x, halfG) - 0.5 * KW;
    const double gy = fma(jj, d.y, halfG) - 0.5 * KW;
    const float dx = (float)(ceil(gx) - gx);
    const float dy = (float)(ceil(gy) - gy);
#if RADON_KB_LUT
    lut_weights(lut, dx, tp.wx);
    lut_weights(lut, dy, tp.wy);
#else
    kb_poly_weights(kp, dx, tp.wx);
    kb_poly_weights(kp, dy, tp.wy);
#endif
}

__device__ __forceinline__ void load_lut_to_smem(float *s_lut, const float *__restrict__ g_lut)
{
#if !RADON_KB_LUT
    return;
#endif
    const float4 *src = reinterpret_cast<const float4 *>(g_lut);
    float4 *dst = reinterpret_cast<float4 *>(s_lut);
    for (int i = threadIdx.x; i < LUT_S * LUT_ROW / 4; i += blockDim.x) dst[i] = __ldg(&src[i]);
}

// =====================================================================================
// F3: inverse gridding (gather)
// =====================================================================================
constexpr int GATHER_THREADS = GATHER_WARPS * 32;
constexpr size_t LUT_SMEM = RADON_KB_LUT ? (size_t)LUT_S * LUT_ROW * sizeof(float) : 0;
constexpr size_t GATHER_SMEM = (size_t)GT_ROWS * GT_PITCH * sizeof(float2) + LUT_SMEM;

__global__ void __launch_bounds__(GATHER_THREADS, 2)
gather_kernel(const float2 *__restrict__ grid, float2 *__restrict__ polar,
              const GatherCta *__restrict__ ctas, const Slot *__restrict__ slots,
              const double2 *__restrict__ cs, const float *__restrict__ g_lut, const KbPoly kp,
              int G, int n_det)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float *s_lut = reinterpret_cast<float *>(smem_raw);
    float2 *tile = reinterpret_cast<float2 *>(smem_raw + LUT_SMEM);

    const GatherCta cta = ctas[blockIdx.x];
    load_lut_to_smem(s_lut, g_lut);

    // stage the tile (+KH halo up/right), indices wrap mod G
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int ly = warp; ly < GT_ROWS; ly += GATHER_WARPS) {
        int gy = cta.ty0 + ly;
        gy = gy % G;
        const float2 *src = grid + (size_t)gy * G;
        for (int lx = lane; lx < GT_PITCH; lx += 32) {
            int gx = cta.tx0 + lx;
            gx = gx % G;
            tile[ly * GT_PITCH + lx] = __ldg(&src[gx]);
        }
    }
    __syncthreads();

    const int cd = n_det / 2;
    const double halfG = 0.5 * (double)G;
    for (int r = warp; r < cta.round_count; r += GATHER_WARPS) {
        const Slot sl = slots[(size_t)(cta.round_begin + r) * 32 + lane];
        if (sl.ak == SLOT_EMPTY) continue;
        const int a = sl.ak >> 16, k = sl.ak & 0xffff;
        Taps tp;
        sample_taps(cs, s_lut, kp, a, k, cd, halfG, tp);
        const float2 *base = tile + (sl.lxy >> 16) * GT_PITCH + (sl.lxy & 0xffff);
        float accr = 0.f, acci = 0.f;
#pragma unroll
        for (int ly = 0; ly < KW; ++ly) {
            float rr = 0.f, ri = 0.f;
#pragma unroll
            for (int lx = 0; lx < KW; ++lx) {
                const float2 v = base[ly * GT_PITCH + lx];
                rr = fmaf(v.x, tp.wx[lx], rr);
                ri = fmaf(v.y, tp.wx[lx], ri);
            }
            accr = fmaf(rr, tp.wy[ly], accr);
            acci = fmaf(ri, tp.wy[ly], acci);
        }
        polar[(size_t)a * n_det + k] = make_float2(accr, acci);
    }
}

// =====================================================================================
// A2: gridding (scatter) -- warp-private accumulators, conflict-free rounds, fixed-order merge
// =====================================================================================
constexpr int SCATTER_THREADS = SCATTER_ITEMS * 32;
constexpr int SP_CELLS = SP_H * SP_PITCH;
constexpr size_t SCATTER_SMEM = (size_t)SCATTER_ITEMS * SP_CELLS * sizeof(float2) + LUT_SMEM;

__global__ void __launch_bounds__(SCATTER_THREADS, 2)
scatter_kernel(const float2 *__restrict__ polar, float2 *__restrict__ grid, float2 *__restrict__ scratch,
               const ScatterCta *__restrict__ ctas, const Slot *__restrict__ slots,
               const double2 *__restrict__ cs, const float *__restrict__ g_lut, const KbPoly kp,
               int G, int n_det)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float *s_lut = reinterpret_cast<float *>(smem_raw);
    float2 *priv = reinterpret_cast<float2 *>(smem_raw + LUT_SMEM);
    __shared__ ScatterCta cta;

    if (threadIdx.x < sizeof(ScatterCta) / 4)
        reinterpret_cast<int *>(&cta)[threadIdx.x] = reinterpret_cast<const int *>(&ctas[blockIdx.x])[threadIdx.x];
    load_lut_to_smem(s_lut, g_lut);
    {
        float4 *z = reinterpret_cast<float4 *>(priv);
        for (int i = threadIdx.x; i < SCATTER_ITEMS * SP_CELLS / 2; i += SCATTER_THREADS)
            z[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    __syncthreads();

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int cd = n_det / 2;
    const double halfG = 0.5 * (double)G;
    {
        const ScatterItem item = cta.items[warp];
        float2 *mine = priv + warp * SP_CELLS;
        for (int r = 0; r < item.round_count; ++r) {
            const Slot sl = slots[(size_t)(item.round_begin + r) * 32 + lane];
            if (sl.ak != SLOT_EMPTY) {
                const int a = sl.ak >> 16, k = sl.ak & 0xffff;
                Taps tp;
                sample_taps(cs, s_lut, kp, a, k, cd, halfG, tp);
                const float2 val = __ldg(&polar[(size_t)a * n_det + k]);
                float2 *base = mine + (sl.lxy >> 16) * SP_PITCH + (sl.lxy & 0xffff);
#pragma unroll
                for (int ly = 0; ly < KW; ++ly) {
                    const float vr = val.x * tp.wy[ly], vi = val.y * tp.wy[ly];
#pragma unroll
                    for (int lx = 0; lx < KW; ++lx) {
                        float2 c = base[ly * SP_PITCH + lx];
                        c.x = fmaf(vr, tp.wx[lx], c.x);
                        c.y = fmaf(vi, tp.wx[lx], c.y);
                        base[ly * SP_PITCH + lx] = c;
                    }
                }
            }
            __syncwarp();   // footprints of one round are disjoint; rounds must not overlap in time
        }
    }
    __syncthreads();

    // merge the warps' accumulators in warp order and write the rectangle exactly once
    float2 *dst;
    int dpitch;
    if (cta.partial_slot >= 0) { dst = scratch + (size_t)cta.partial_slot * (ST_X * ST_Y); dpitch = ST_X; }
    else { dst = grid + (size_t)cta.ry0 * G + cta.rx0; dpitch = G; }
    const int cells = cta.rw * cta.rh;
    for (int i = threadIdx.x; i < cells; i += SCATTER_THREADS) {
        const int y = i / cta.rw, x = i - y * cta.rw;
        float sr = 0.f, si = 0.f;
#pragma unroll
        for (int it = 0; it < SCATTER_ITEMS; ++it) {
            const int lx = cta.rx0 + x - cta.items[it].px0, ly = cta.ry0 + y - cta.items[it].py0;
            if (cta.items[it].round_count > 0 && (unsigned)lx < (unsigned)SP_W && (unsigned)ly < (unsigned)SP_H) {
                const float2 c = priv[it * SP_CELLS + ly * SP_PITCH + lx];
                sr += c.x;
                si += c.y;
            }
        }
        dst[(size_t)y * dpitch + x] = make_float2(sr, si);
    }
}

__global__ void __launch_bounds__(256)
merge_kernel(const float2 *__restrict__ scratch, float2 *__restrict__ grid,
             const MergeJob *__restrict__ jobs, int G)
{
    const MergeJob j = jobs[blockIdx.x];
    for (int i = threadIdx.x; i < j.rw * j.rh; i += blockDim.x) {
        const int y = i / j.rw, x = i - y * j.rw;
        float sr = 0.f, si = 0.f;
        for (int s = 0; s < j.n_slots; ++s) {
            const float2 c = scratch[(size_t)(j.first_slot + s) * (ST_X * ST_Y) + y * ST_X + x];
            sr += c.x;
            si += c.y;
        }
        grid[(size_t)(j.ry0 + y) * G + j.rx0 + x] = make_float2(sr, si);
    }
}

int launch_gather(const DevicePlan &p, const float2 *grid, float2 *polar, cudaStream_t st)
{
    if (p.n_gather_ctas == 0) return 0;
    gather_kernel<<<p.n_gather_ctas, GATHER_THREADS, GATHER_SMEM, st>>>(
        grid, polar, p.gather_ctas, p.gather_slots, p.cs, p.lut, p.kb, p.G, p.n_det);
    count_launch();
    return 0;
}

int launch_scatter(const DevicePlan &p, const float2 *polar, float2 *grid, cudaStream_t st)
{
    scatter_kernel<<<p.n_scatter_ctas, SCATTER_THREADS, SCATTER_SMEM, st>>>(
        polar, grid, p.scratch, p.scatter_ctas, p.scatter_slots, p.cs, p.lut, p.kb, p.G, p.n_det);
    count_launch();
    if (p.n_merge_jobs > 0) {
        merge_kernel<<<p.n_merge_jobs, 256, 0, st>>>(p.scratch, grid, p.merge_jobs, p.G);
        count_launch();
    }
    return 0;
}

int init_kernel_attributes()
{
    if (set_smem(gather_kernel, GATHER_SMEM)) return -1;
    if (set_smem(scatter_kernel, SCATTER_SMEM)) return -1;
    return 0;
}

}  // namespace radon
