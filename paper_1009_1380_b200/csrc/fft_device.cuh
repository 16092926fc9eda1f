// fft_device.cuh -- shared-memory Stockham FFT for power-of-two lengths 16 .. 8192.
//
// No cuFFT (BASELINE.json north_star: "shared-memory radix 2D FFT of the oversampled image
// and batched 1D FFTs along each projection").  One FFT of length L is computed by L/16
// threads; every thread keeps 16 complex values in registers per pass and performs
// radix-16 butterflies (one radix-2/4/8 pass first when log2 L is not a multiple of 4).
// Data live in shared memory between passes, skewed by one element per 16 (FFT_PAD) so that
// the stride-16 writes of the first pass do not collide in one bank pair.
// Twiddles exp(-2 pi i q / L) come from a table derived in fp64 at plan time.
#pragma once
#include <cuda_runtime.h>

namespace radon {

#define FFT_PAD(i) ((i) + ((i) >> 4))
__host__ __device__ constexpr int fft_padded_len(int L) { return L + (L >> 4); }

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
// a * w (SIGN < 0, forward) or a * conj(w) (SIGN > 0, inverse); w = exp(-i phi)
template <int SIGN>
__device__ __forceinline__ float2 cmul_tw(float2 a, float2 w)
{
    if (SIGN < 0) return make_float2(fmaf(a.x, w.x, -a.y * w.y), fmaf(a.x, w.y, a.y * w.x));
    return make_float2(fmaf(a.x, w.x, a.y * w.y), fmaf(-a.x, w.y, a.y * w.x));
}

// exp(-2 pi i k / 16), k = 0..7, folded to constants after unrolling
__device__ __forceinline__ float2 tw16(int k)
{
    constexpr float c[8] = {1.0f, 0.92387953251128674f, 0.70710678118654752f, 0.38268343236508977f,
                            0.0f, -0.38268343236508977f, -0.70710678118654752f, -0.92387953251128674f};
    constexpr float s[8] = {0.0f, 0.38268343236508977f, 0.70710678118654752f, 0.92387953251128674f,
                            1.0f, 0.92387953251128674f, 0.70710678118654752f, 0.38268343236508977f};
    return make_float2(c[k], -s[k]);
}

// In-register DFT of R points, natural order in and out.
template <int R, int SIGN>
__device__ __forceinline__ void dft_reg(float2 (&v)[R])
{
    if constexpr (R == 1) {
        return;
    } else if constexpr (R == 2) {
        const float2 a = v[0], b = v[1];
        v[0] = cadd(a, b);
        v[1] = csub(a, b);
    } else if constexpr (R == 4) {
        const float2 t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]);
        const float2 t2 = cadd(v[1], v[3]), t3 = csub(v[1], v[3]);
        v[0] = cadd(t0, t2);
        v[2] = csub(t0, t2);
        if (SIGN < 0) {   // multiply t3 by -i
            v[1] = make_float2(t1.x + t3.y, t1.y - t3.x);
            v[3] = make_float2(t1.x - t3.y, t1.y + t3.x);
        } else {          // multiply t3 by +i
            v[1] = make_float2(t1.x - t3.y, t1.y + t3.x);
            v[3] = make_float2(t1.x + t3.y, t1.y - t3.x);
        }
    } else {
        float2 e[R / 2], o[R / 2];
#pragma unroll
        for (int i = 0; i < R / 2; ++i) { e[i] = v[2 * i]; o[i] = v[2 * i + 1]; }
        dft_reg<R / 2, SIGN>(e);
        dft_reg<R / 2, SIGN>(o);
#pragma unroll
        for (int k = 0; k < R / 2; ++k) {
            const float2 t = cmul_tw<SIGN>(o[k], tw16(k * (16 / R)));
            v[k] = cadd(e[k], t);
            v[k + R / 2] = csub(e[k], t);
        }
    }
}

// One Stockham pass of radix R with NS = product of the radices already applied.
template <int L, int R, int NS, int SIGN>
__device__ __forceinline__ void fft_pass(float2 *s, const float2 *__restrict__ tw, int t)
{
    constexpr int TF = L / 16, NB = 16 / R, STRIDE = L / R;
    float2 v[NB][R];
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        const int j = b * TF + t;
#pragma unroll
        for (int q = 0; q < R; ++q) v[b][q] = s[FFT_PAD(j + q * STRIDE)];
    }
    __syncthreads();
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        const int j = b * TF + t;
        const int jm = j & (NS - 1);
        if (NS > 1) {
#pragma unroll
            for (int q = 1; q < R; ++q) {
                const float2 w = __ldg(&tw[jm * q * (L / (NS * R))]);
                v[b][q] = cmul_tw<SIGN>(v[b][q], w);
            }
        }
        dft_reg<R, SIGN>(v[b]);
        const int base = (j - jm) * R + jm;
#pragma unroll
        for (int u = 0; u < R; ++u) s[FFT_PAD(base + u * NS)] = v[b][u];
    }
    __syncthreads();
}

__host__ __device__ constexpr int ilog2_c(int v) { return v <= 1 ? 0 : 1 + ilog2_c(v >> 1); }

// Length-L FFT (SIGN<0: forward exp(-i..), SIGN>0: unnormalised inverse) of the padded
// shared-memory array s by threads t = 0 .. L/16-1.  Every thread of the CTA must call it
// (it contains __syncthreads); the caller synchronises after filling s.
template <int L, int SIGN>
__device__ __forceinline__ void fft_smem(float2 *s, const float2 *__restrict__ tw, int t)
{
    constexpr int LOG = ilog2_c(L);
    constexpr int R0 = 1 << (LOG % 4);          // first pass: radix 1 (none), 2, 4 or 8
    constexpr int NQ = LOG / 4;                 // then NQ radix-16 passes
    if constexpr (R0 > 1) fft_pass<L, R0, 1, SIGN>(s, tw, t);
    if constexpr (NQ >= 1) fft_pass<L, 16, R0, SIGN>(s, tw, t);
    if constexpr (NQ >= 2) fft_pass<L, 16, R0 * 16, SIGN>(s, tw, t);
    if constexpr (NQ >= 3) fft_pass<L, 16, R0 * 256, SIGN>(s, tw, t);
}

}  // namespace radon
