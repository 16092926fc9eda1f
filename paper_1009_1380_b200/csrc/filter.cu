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

// ---- axis 0: one CTA per projection ----------------------------------------------------------
constexpr int FROW_THREADS = 256;
__global__ void __launch_bounds__(FROW_THREADS)
filter_rows_kernel(const float *__restrict__ in, float *__restrict__ out, const float *__restrict__ q, int n, int hi)
{
    __shared__ float part[FROW_THREADS / 32][FILTER_MAXQ];
    pdl_prologue();
    const float *z = in + (size_t)blockIdx.x * n;
    float c[FILTER_MAXQ];
#pragma unroll
    for (int d = 0; d < FILTER_MAXQ; ++d) c[d] = 0.f;
    for (int s0 = threadIdx.x; s0 < n; s0 += 4 * FROW_THREADS) {        // four elements (twelve loads) in flight
        float v[4];
        float4 qa[4], qb[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int s = min(s0 + u * FROW_THREADS, n - 1);
            v[u] = (s0 + u * FROW_THREADS < n) ? __ldg(&z[s]) : 0.f;
            qa[u] = __ldg(reinterpret_cast<const float4 *>(q + (size_t)s * FILTER_MAXQ));
            qb[u] = hi ? __ldg(reinterpret_cast<const float4 *>(q + (size_t)s * FILTER_MAXQ + 4)) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            c[0] = fmaf(qa[u].x, v[u], c[0]); c[1] = fmaf(qa[u].y, v[u], c[1]); c[2] = fmaf(qa[u].z, v[u], c[2]); c[3] = fmaf(qa[u].w, v[u], c[3]);
            c[4] = fmaf(qb[u].x, v[u], c[4]); c[5] = fmaf(qb[u].y, v[u], c[5]); c[6] = fmaf(qb[u].z, v[u], c[6]); c[7] = fmaf(qb[u].w, v[u], c[7]);
        }
    }
#pragma unroll
    for (int d = 0; d < FILTER_MAXQ; ++d)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) c[d] += __shfl_xor_sync(0xffffffffu, c[d], o);
    if ((threadIdx.x & 31) == 0)
#pragma unroll
        for (int d = 0; d < FILTER_MAXQ; ++d) part[threadIdx.x >> 5][d] = c[d];
    __syncthreads();
#pragma unroll
    for (int d = 0; d < FILTER_MAXQ; ++d) {
        float a = 0.f;
        for (int w = 0; w < FROW_THREADS / 32; ++w) a += part[w][d];        // fixed order
        c[d] = a;
    }
    pdl_trigger();
    float *o_row = out + (size_t)blockIdx.x * n;
    for (int s = threadIdx.x; s < n; s += FROW_THREADS) {
        const float4 qa = __ldg(reinterpret_cast<const float4 *>(q + (size_t)s * FILTER_MAXQ));
        const float4 qb = hi ? __ldg(reinterpret_cast<const float4 *>(q + (size_t)s * FILTER_MAXQ + 4)) : make_float4(0.f, 0.f, 0.f, 0.f);
        float fit = qa.x * c[0];
        fit = fmaf(qa.y, c[1], fit); fit = fmaf(qa.z, c[2], fit); fit = fmaf(qa.w, c[3], fit);
        fit = fmaf(qb.x, c[4], fit); fit = fmaf(qb.y, c[5], fit); fit = fmaf(qb.z, c[6], fit); fit = fmaf(qb.w, c[7], fit);
        o_row[s] = __ldg(&z[s]) - fit;       // rows of q beyond the order are zero
    }
}

// ---- axis 1: a CTA owns FCOL_COLS adjacent detector bins (one 32-byte sector per sinogram row),
//      FCOL_PARTS threads per bin split the angles -------------------------------------------------
constexpr int FCOL_COLS = 8, FCOL_PARTS = 64;
__global__ void __launch_bounds__(FCOL_COLS * FCOL_PARTS)
filter_cols_kernel(const float *__restrict__ in, float *__restrict__ out, const float *__restrict__ q,
                   int n_cols, int n_rows, int hi)
{
    __shared__ float part[FCOL_PARTS][FILTER_MAXQ][FCOL_COLS + 1];
    pdl_prologue();
    const int lc = threadIdx.x % FCOL_COLS, pr = threadIdx.x / FCOL_COLS;
    const int col = blockIdx.x * FCOL_COLS + lc;
    const bool live = col < n_cols;
    float c[FILTER_MAXQ];
#pragma unroll
    for (int d = 0; d < FILTER_MAXQ; ++d) c[d] = 0.f;
    for (int a0 = pr; a0 < n_rows; a0 += 4 * FCOL_PARTS) {
        float v[4];
        float4 qa[4], qb[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int a = min(a0 + u * FCOL_PARTS, n_rows - 1);
            v[u] = (live && a0 + u * FCOL_PARTS < n_rows) ? __ldg(&in[(size_t)a * n_cols + col]) : 0.f;
            qa[u] = __ldg(reinterpret_cast<const float4 *>(q + (size_t)a * FILTER_MAXQ));
            qb[u] = hi ? __ldg(reinterpret_cast<const float4 *>(q + (size_t)a * FILTER_MAXQ + 4)) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            c[0] = fmaf(qa[u].x, v[u], c[0]); c[1] = fmaf(qa[u].y, v[u], c[1]); c[2] = fmaf(qa[u].z, v[u], c[2]); c[3] = fmaf(qa[u].w, v[u], c[3]);
            c[4] = fmaf(qb[u].x, v[u], c[4]); c[5] = fmaf(qb[u].y, v[u], c[5]); c[6] = fmaf(qb[u].z, v[u], c[6]); c[7] = fmaf(qb[u].w, v[u], c[7]);
        }
    }
#pragma unroll
    for (int d = 0; d < FILTER_MAXQ; ++d) part[pr][d][lc] = c[d];
    __syncthreads();
#pragma unroll
    for (int d = 0; d < FILTER_MAXQ; ++d) {
        float s = 0.f;
        for (int p = 0; p < FCOL_PARTS; ++p) s += part[p][d][lc];     // fixed order
        c[d] = s;
    }
    pdl_trigger();
    if (!live) return;
    for (int a = pr; a < n_rows; a += FCOL_PARTS) {
        const float4 qa = __ldg(reinterpret_cast<const float4 *>(q + (size_t)a * FILTER_MAXQ));
        const float4 qb = hi ? __ldg(reinterpret_cast<const float4 *>(q + (size_t)a * FILTER_MAXQ + 4)) : make_float4(0.f, 0.f, 0.f, 0.f);
        float fit = qa.x * c[0];
        fit = fmaf(qa.y, c[1], fit); fit = fmaf(qa.z, c[2], fit); fit = fmaf(qa.w, c[3], fit);
        fit = fmaf(qb.x, c[4], fit); fit = fmaf(qb.y, c[5], fit); fit = fmaf(qb.z, c[6], fit); fit = fmaf(qb.w, c[7], fit);
        out[(size_t)a * n_cols + col] = __ldg(&in[(size_t)a * n_cols + col]) - fit;
    }
}

int launch_filter(const DevicePlan &p, int axis, const float *q, int order, const float *in, float *out, cudaStream_t st)
{
    if (axis == 0)
        launch_pdl(p.pdl, filter_rows_kernel, p.n_angles, FROW_THREADS, 0, st, in, out, q, p.n_det, order > 3 ? 1 : 0);
    else
        launch_pdl(p.pdl, filter_cols_kernel, (p.n_det + FCOL_COLS - 1) / FCOL_COLS, FCOL_COLS * FCOL_PARTS, 0, st, in, out, q, p.n_det, p.n_angles, order > 3 ? 1 : 0);
    count_launch();
    return 0;
}

}  // namespace radon
