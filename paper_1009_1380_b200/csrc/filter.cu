// filter.cu -- the sinogram filter of the paper's objective, filter(Radon{x} - data)
// (PAPER.md:31, :47): "a 3rd order polynomial fit to smooth the sinogram and reduce the ringing
// artifacts", applied as "polynomial subtraction".  Reading R-filter
// (DESIGN.md section 4): along one axis of the sinogram the least-squares polynomial of degree
// p is subtracted, z <- z - sum_d q_d <q_d, z>, with q_0..q_p the orthonormal discrete
// polynomials on the line's sample points (built in fp64 at plan time, plan_host.cpp).  The
// operator is an orthogonal projector: symmetric and idempotent.
//   axis 0: along the detector coordinate of every projection (the fluctuation of the
//           illuminating beam from exposure to exposure) -- also fused into the
//           projection DFT kernels (proj.cu) for radon_forward_filtered / radon_adjoint_filtered;
//   axis 1: along the angle coordinate of every detector bin.
#include "kernels.h"

namespace radon {

// ---- axis 0: one warp per projection -------------------------------------------------------
constexpr int FROW_WARPS = 8;
__global__ void __launch_bounds__(FROW_WARPS * 32)
filter_rows_kernel(const float *__restrict__ in, float *__restrict__ out, const float *__restrict__ q,
                   int n, int n_rows, int nq)
{
    const int row = blockIdx.x * FROW_WARPS + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (row >= n_rows) return;
    const float *z = in + (size_t)row * n;
    float c[FILTER_MAXQ];
#pragma unroll
    for (int d = 0; d < FILTER_MAXQ; ++d) c[d] = 0.f;
    for (int s = lane; s < n; s += 32) {
        const float v = __ldg(&z[s]);
        const float4 qa = __ldg(reinterpret_cast<const float4 *>(q + (size_t)s * FILTER_MAXQ));
        const float4 qb = __ldg(reinterpret_cast<const float4 *>(q + (size_t)s * FILTER_MAXQ + 4));
        c[0] = fmaf(qa.x, v, c[0]); c[1] = fmaf(qa.y, v, c[1]); c[2] = fmaf(qa.z, v, c[2]); c[3] = fmaf(qa.w, v, c[3]);
        c[4] = fmaf(qb.x, v, c[4]); c[5] = fmaf(qb.y, v, c[5]); c[6] = fmaf(qb.z, v, c[6]); c[7] = fmaf(qb.w, v, c[7]);
    }
#pragma unroll
    for (int d = 0; d < FILTER_MAXQ; ++d)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) c[d] += __shfl_xor_sync(0xffffffffu, c[d], o);
    float *o_row = out + (size_t)row * n;
    for (int s = lane; s < n; s += 32) {
        const float4 qa = __ldg(reinterpret_cast<const float4 *>(q + (size_t)s * FILTER_MAXQ));
        const float4 qb = __ldg(reinterpret_cast<const float4 *>(q + (size_t)s * FILTER_MAXQ + 4));
        float fit = qa.x * c[0];
        fit = fmaf(qa.y, c[1], fit); fit = fmaf(qa.z, c[2], fit); fit = fmaf(qa.w, c[3], fit);
        fit = fmaf(qb.x, c[4], fit); fit = fmaf(qb.y, c[5], fit); fit = fmaf(qb.z, c[6], fit); fit = fmaf(qb.w, c[7], fit);
        o_row[s] = __ldg(&z[s]) - fit;       // rows of q beyond the order are zero
    }
    (void)nq;
}

// ---- axis 1: a CTA owns 32 adjacent detector bins, FCOL_PARTS threads per bin split the angles ----
constexpr int FCOL_PARTS = 16;
__global__ void __launch_bounds__(32 * FCOL_PARTS)
filter_cols_kernel(const float *__restrict__ in, float *__restrict__ out, const float *__restrict__ q,
                   int n_cols, int n_rows)
{
    __shared__ float part[FCOL_PARTS][FILTER_MAXQ][33];
    const int col = blockIdx.x * 32 + (threadIdx.x & 31), pr = threadIdx.x >> 5;
    const bool live = col < n_cols;
    float c[FILTER_MAXQ];
#pragma unroll
    for (int d = 0; d < FILTER_MAXQ; ++d) c[d] = 0.f;
    for (int a = pr; a < n_rows; a += FCOL_PARTS) {
        const float v = live ? __ldg(&in[(size_t)a * n_cols + col]) : 0.f;
        const float4 qa = __ldg(reinterpret_cast<const float4 *>(q + (size_t)a * FILTER_MAXQ));   // warp-uniform
        const float4 qb = __ldg(reinterpret_cast<const float4 *>(q + (size_t)a * FILTER_MAXQ + 4));
        c[0] = fmaf(qa.x, v, c[0]); c[1] = fmaf(qa.y, v, c[1]); c[2] = fmaf(qa.z, v, c[2]); c[3] = fmaf(qa.w, v, c[3]);
        c[4] = fmaf(qb.x, v, c[4]); c[5] = fmaf(qb.y, v, c[5]); c[6] = fmaf(qb.z, v, c[6]); c[7] = fmaf(qb.w, v, c[7]);
    }
#pragma unroll
    for (int d = 0; d < FILTER_MAXQ; ++d) part[pr][d][threadIdx.x & 31] = c[d];
    __syncthreads();
#pragma unroll
    for (int d = 0; d < FILTER_MAXQ; ++d) {
        float s = 0.f;
        for (int p = 0; p < FCOL_PARTS; ++p) s += part[p][d][threadIdx.x & 31];     // fixed order
        c[d] = s;
    }
    if (!live) return;
    for (int a = pr; a < n_rows; a += FCOL_PARTS) {
        const float4 qa = __ldg(reinterpret_cast<const float4 *>(q + (size_t)a * FILTER_MAXQ));
        const float4 qb = __ldg(reinterpret_cast<const float4 *>(q + (size_t)a * FILTER_MAXQ + 4));
        float fit = qa.x * c[0];
        fit = fmaf(qa.y, c[1], fit); fit = fmaf(qa.z, c[2], fit); fit = fmaf(qa.w, c[3], fit);
        fit = fmaf(qb.x, c[4], fit); fit = fmaf(qb.y, c[5], fit); fit = fmaf(qb.z, c[6], fit); fit = fmaf(qb.w, c[7], fit);
        out[(size_t)a * n_cols + col] = __ldg(&in[(size_t)a * n_cols + col]) - fit;
    }
}

int launch_filter(const DevicePlan &p, int axis, const float *q, const float *in, float *out, cudaStream_t st)
{
    if (axis == 0)
        filter_rows_kernel<<<(p.n_angles + FROW_WARPS - 1) / FROW_WARPS, FROW_WARPS * 32, 0, st>>>(in, out, q, p.n_det, p.n_angles, 0);
    else
        filter_cols_kernel<<<(p.n_det + 31) / 32, 32 * FCOL_PARTS, 0, st>>>(in, out, q, p.n_det, p.n_angles);
    count_launch();
    return 0;
}

}  // namespace radon
