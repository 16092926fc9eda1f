// fft2d_composite.cu -- the four 2-D FFT passes of the path (fft2d.cu) for oversampled grid sides
// that are not a power of two: L = 3 * 2^m or 5 * 2^m (N = 1536 or 2560 at sigma = 2, ...).
//
// One decimation-in-time step in front of the power-of-two Stockham FFT of fft_device.cuh:
//   x_r[n] = x[PR n + r],  F_r = FFT_P(x_r),  r = 0 .. PR-1,  L = PR * P,
//   X[k + q P] = sum_r F_r[k] W_L^{r (k + q P)}           (W_L = exp(-+ 2 pi i / L)).
// Thread (r, t) of a line's L/16 threads holds x_r[t + i P/16] on entry, runs fft_reg<P> with the
// other P/16 - 1 threads of its group r, and after one exchange through shared memory leaves with
// X[t + i P/16 + r P], i = 0 .. 15: contiguous blocks on both sides of the global memory traffic.
// Plain versions of the passes (one real column per line in the column passes, no packed pairs,
// no staging by the copy engine): the layouts of T and of the grid are those of fft2d.cu, so the
// gridding kernels and the projection kernels do not see the difference.
#include "kernels.h"

#include "fft_device.cuh"

namespace radon {

template <int P, int PR>
struct CompCfg {
    static constexpr int L = P * PR;
    static constexpr int TF = P / 16;                     // threads per sub-FFT
    static constexpr int THREADS = PR * TF;               // threads per line
    static constexpr int PADLEN = fft_padded_len(P);
    static constexpr size_t SMEM = (size_t)PR * PADLEN * sizeof(float2);
};

__device__ __forceinline__ int emod(int v, int L)
{
    v %= L;
    return v < 0 ? v + L : v;
}

// in : v[i] = x[PR (t + i TF) + r];  out: v[i] = X[t + i TF + r P].  s_all: PR * PADLEN float2.
// twP: exp(-2 pi i q / P), twL: exp(-2 pi i q / L).  Every thread of the CTA calls it.
template <int P, int PR, int SIGN>
__device__ __forceinline__ void fft_composite(float2 (&v)[16], float2 *s_all, const float2 *__restrict__ twP,
                                              const float2 *__restrict__ twL, int t, int r)
{
    using C = CompCfg<P, PR>;
    float2 *s = s_all + r * C::PADLEN;
    fft_reg<P, SIGN>(v, s, twP, t);
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 16; ++i) s[FFT_PAD(t + i * C::TF)] = v[i];
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int k = t + i * C::TF, o = k + r * P;
        float2 acc = s_all[FFT_PAD(k)];                    // r' = 0: W^0
#pragma unroll
        for (int rr = 1; rr < PR; ++rr) {
            const float2 f = s_all[rr * C::PADLEN + FFT_PAD(k)];
            const float2 w = __ldg(&twL[(int)(((long long)rr * o) % C::L)]);
            const float2 p = cmul_tw<SIGN>(f, w);
            acc.x += p.x; acc.y += p.y;
        }
        v[i] = acc;
    }
    __syncthreads();
}

// ---- F1 + columns of F2: one real image column per CTA --------------------------------------------
template <int P, int PR>
__global__ void __launch_bounds__(CompCfg<P, PR>::THREADS)
colpass_fwd_comp_kernel(const float *__restrict__ x, const float *__restrict__ deapod, float2 *__restrict__ T,
                        const float2 *__restrict__ twP, const float2 *__restrict__ twL, int N)
{
    extern __shared__ __align__(16) float2 s_fft[];
    using C = CompCfg<P, PR>;
    pdl_prologue();
    const int r = threadIdx.x / C::TF, t = threadIdx.x - r * C::TF, ix = blockIdx.x, c = N / 2;
    const float da = __ldg(&deapod[ix]);
    float2 v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int iy = emod(PR * (t + i * C::TF) + r + c, C::L);          // FFT position (iy - c) mod L
        v[i] = make_float2(iy < N ? __ldg(&x[(size_t)iy * N + ix]) * da * __ldg(&deapod[iy]) : 0.f, 0.f);
    }
    fft_composite<P, PR, -1>(v, s_fft, twP, twL, t, r);
    pdl_trigger();
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int k = t + i * C::TF + r * P;
        if (k <= C::L / 2) T[(size_t)k * N + ix] = v[i];                  // Hermitian half of a real column
    }
}

// ---- rows of F2: T row ky -> centred grid row ky (and its mirror) ---------------------------------------
template <int P, int PR>
__global__ void __launch_bounds__(CompCfg<P, PR>::THREADS)
rowpass_fwd_comp_kernel(const float2 *__restrict__ T, float2 *__restrict__ grid, const float2 *__restrict__ twP,
                        const float2 *__restrict__ twL, int N, int mirror, int KW)
{
    extern __shared__ __align__(16) float2 s_fft[];
    using C = CompCfg<P, PR>;
    constexpr int L = C::L;
    pdl_prologue();
    const int r = threadIdx.x / C::TF, t = threadIdx.x - r * C::TF, ky = blockIdx.x, c = N / 2;
    float2 v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int ix = emod(PR * (t + i * C::TF) + r + c, L);
        v[i] = ix < N ? __ldg(&T[(size_t)ky * N + ix]) : make_float2(0.f, 0.f);
    }
    fft_composite<P, PR, -1>(v, s_fft, twP, twL, t, r);
    pdl_trigger();
    const int cy = emod(ky + L / 2, L);
    float2 *row = grid + (size_t)cy * L;
#pragma unroll
    for (int i = 0; i < 16; ++i) row[emod(t + i * C::TF + r * P + L / 2, L)] = v[i];
    const bool want = mirror == 1 || (mirror == 2 && (ky <= KW / 2 || ky >= L / 2 - (KW / 2 - 1)));
    if (want && ky != 0 && ky != L / 2) {
        float2 *mrow = grid + (size_t)(L - cy) * L;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const int cx = emod(t + i * C::TF + r * P + L / 2, L);
            mrow[emod(L - cx, L)] = cconj(v[i]);
        }
    }
}

// ---- rows of A3: grid row ky (Hermitian part when fold) -> T ---------------------------------------------
template <int P, int PR>
__global__ void __launch_bounds__(CompCfg<P, PR>::THREADS)
rowpass_inv_comp_kernel(const float2 *__restrict__ grid, float2 *__restrict__ T, const float2 *__restrict__ twP,
                        const float2 *__restrict__ twL, int N, int fold)
{
    extern __shared__ __align__(16) float2 s_fft[];
    using C = CompCfg<P, PR>;
    constexpr int L = C::L;
    pdl_prologue();
    const int r = threadIdx.x / C::TF, t = threadIdx.x - r * C::TF, ky = blockIdx.x, c = N / 2;
    const int cy = emod(ky + L / 2, L);
    const float2 *row = grid + (size_t)cy * L, *mrow = grid + (size_t)emod(L - cy, L) * L;
    float2 v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int cx = emod(PR * (t + i * C::TF) + r + L / 2, L);
        v[i] = __ldg(&row[cx]);
        if (fold) {
            const float2 w = __ldg(&mrow[emod(L - cx, L)]);
            v[i] = make_float2(0.5f * (v[i].x + w.x), 0.5f * (v[i].y - w.y));
        }
    }
    fft_composite<P, PR, +1>(v, s_fft, twP, twL, t, r);
    pdl_trigger();
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int ix = emod(t + i * C::TF + r * P + c, L);
        if (ix < N) T[(size_t)ky * N + ix] = v[i];
    }
}

// ---- columns of A3 + A4: one image column per CTA ---------------------------------------------------------
template <int P, int PR>
__global__ void __launch_bounds__(CompCfg<P, PR>::THREADS)
colpass_inv_comp_kernel(const float2 *__restrict__ T, const float *__restrict__ deapod, float *x,
                        const float2 *__restrict__ twP, const float2 *__restrict__ twL, int N,
                        int update, float alpha, float tau)
{
    extern __shared__ __align__(16) float2 s_fft[];
    using C = CompCfg<P, PR>;
    constexpr int L = C::L;
    pdl_prologue();
    const int r = threadIdx.x / C::TF, t = threadIdx.x - r * C::TF, ix = blockIdx.x, c = N / 2;
    float2 v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int k = PR * (t + i * C::TF) + r;                           // Hermitian completion of the stored half
        if (k <= L / 2) {
            v[i] = __ldg(&T[(size_t)k * N + ix]);
            if (k == 0 || k == L / 2) v[i].y = 0.f;                       // real by symmetry
        } else {
            v[i] = cconj(__ldg(&T[(size_t)(L - k) * N + ix]));
        }
    }
    fft_composite<P, PR, +1>(v, s_fft, twP, twL, t, r);
    pdl_trigger();
    const float da = __ldg(&deapod[ix]);
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int iy = emod(t + i * C::TF + r * P + c, L);
        if (iy < N) {
            float g = v[i].x * da * __ldg(&deapod[iy]);
            float *px = x + (size_t)iy * N + ix;
            if (update) {                                                 // solver iteration: x <- S_tau(x - alpha g)
                const float u = fmaf(-alpha, g, *px);
                g = copysignf(fmaxf(fabsf(u) - tau, 0.f), u);
            }
            *px = g;
        }
    }
}

// ---- dispatch -------------------------------------------------------------------------------------------------
bool fft_composite_split(int L, int *P_out, int *PR_out)
{
    for (int pr : {3, 5}) {
        if (L % pr) continue;
        const int P = L / pr;
        if (P >= 16 && P <= 2048 && (P & (P - 1)) == 0) {
            if (P_out) *P_out = P;
            if (PR_out) *PR_out = pr;
            return true;
        }
    }
    return false;
}

template <int P, int PR>
static int comp_launch(int which, const DevicePlan &p, const void *in, void *out, int flag, cudaStream_t st,
                       const IstaUpdate *upd)
{
    using C = CompCfg<P, PR>;
    const int N = p.N;
    const dim3 block(C::THREADS);
    switch (which) {
    case 0:
        if (set_smem(colpass_fwd_comp_kernel<P, PR>, C::SMEM)) return -1;
        launch_pdl(p.pdl, colpass_fwd_comp_kernel<P, PR>, N, block, C::SMEM, st, (const float *)in, p.deapod, (float2 *)out, p.tw_sub, p.tw_G, N);
        break;
    case 1:
        if (set_smem(rowpass_fwd_comp_kernel<P, PR>, C::SMEM)) return -1;
        launch_pdl(p.pdl, rowpass_fwd_comp_kernel<P, PR>, C::L / 2 + 1, block, C::SMEM, st, (const float2 *)in, (float2 *)out, p.tw_sub, p.tw_G, N, flag, p.W);
        break;
    case 2:
        if (set_smem(rowpass_inv_comp_kernel<P, PR>, C::SMEM)) return -1;
        launch_pdl(p.pdl, rowpass_inv_comp_kernel<P, PR>, C::L / 2 + 1, block, C::SMEM, st, (const float2 *)in, (float2 *)out, p.tw_sub, p.tw_G, N, flag);
        break;
    case 3:
        if (set_smem(colpass_inv_comp_kernel<P, PR>, C::SMEM)) return -1;
        launch_pdl(p.pdl, colpass_inv_comp_kernel<P, PR>, N, block, C::SMEM, st, (const float2 *)in, p.deapod, (float *)out, p.tw_sub, p.tw_G, N,
                   upd ? 1 : 0, upd ? upd->alpha : 0.f, upd ? upd->tau : 0.f);
        break;
    default:
        return -1;
    }
    count_launch();
    return 0;
}

#define RADON_COMP_CASE(PP)                                                                  \
    case PP:                                                                                 \
        return PR == 3 ? comp_launch<PP, 3>(which, p, in, out, flag, st, upd)                \
                       : comp_launch<PP, 5>(which, p, in, out, flag, st, upd);

int launch_fft2d_composite(int which, const DevicePlan &p, const void *in, void *out, int flag, cudaStream_t st,
                           const IstaUpdate *upd)
{
    int P = 0, PR = 0;
    if (!fft_composite_split(p.G, &P, &PR)) return -1;
    switch (P) {
        RADON_COMP_CASE(16) RADON_COMP_CASE(32) RADON_COMP_CASE(64) RADON_COMP_CASE(128)
        RADON_COMP_CASE(256) RADON_COMP_CASE(512) RADON_COMP_CASE(1024) RADON_COMP_CASE(2048)
    default:
        return -1;
    }
}

}  // namespace radon
