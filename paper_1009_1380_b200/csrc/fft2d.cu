// fft2d.cu -- F1+F2 (de-apodise, zero-pad, 2-D FFT) and A3+A4 (2-D inverse FFT, crop,
// de-apodise) of the NUFFT-Radon path ("first perform a 2D FFT of x on a regular
// grid"), hand-written for sm_100a, no cuFFT.
//
// The image side of both transforms is REAL, so both are real <-> Hermitian transforms
// ("input real -> r2c/Hermitian halving possible"; row A3: "only N^2
// outputs needed -> prunable"):
//   forward   column pass: two real image columns packed into ONE complex length-G FFT along Y
//             (z = a + i b), untangled through shared memory into the Hermitian halves
//             T[ky][ix], ky = 0..G/2 (zero-padding pruned: only N of G inputs are loaded);
//             row pass: one complex FFT along X per ky = 0..G/2 (N non-zero inputs), written
//             to the centred grid row ky and, conjugate-reversed, to the mirrored row -ky.
//   inverse   row pass: Hermitian part of the grid (G(k) + conj G(-k))/2 for ky = 0..G/2
//             (Re{IFFT2(G)} = IFFT2(Hermitian part of G)), inverse FFT along X, N centre
//             outputs kept -> T; column pass: two columns packed (Z = A + i B), inverse FFT
//             along Y gives a + i b, cropped, de-apodised.
// The strided (column) accesses fall on the small arrays (image, T); every access to the
// 8 G^2-byte grid is a contiguous row.  T = (G/2+1) x N c64 (33.6 MB at config 4) is written
// and read back within one call and stays L2-resident.
#include "kernels.h"
#include "fft_device.cuh"

namespace radon {

template <int L>
struct FftCfg {
    static constexpr int TF = L / 16;                                  // threads per FFT
    static constexpr int NF = (TF >= 128) ? 1 : 128 / TF;              // FFTs per CTA
    static constexpr int THREADS = NF * TF;
    static constexpr int PADLEN = fft_padded_len(L);
    static constexpr size_t SMEM = (size_t)NF * PADLEN * sizeof(float2);
};

// ---- F1 + first half of F2 ------------------------------------------------------------------
template <int L>
__global__ void __launch_bounds__(FftCfg<L>::THREADS)
colpass_fwd_kernel(const float *__restrict__ x, const float *__restrict__ deapod,
                   float2 *__restrict__ T, const float2 *__restrict__ tw, int N)
{
    extern __shared__ __align__(16) float2 s_fft[];
    using C = FftCfg<L>;
    constexpr int TF = C::TF;
    const int f = threadIdx.x / TF, t = threadIdx.x - f * TF;
    float2 *s = s_fft + f * C::PADLEN;
    const int p = blockIdx.x * C::NF + f, ix = 2 * p;
    const bool live = ix < N, has_b = ix + 1 < N;
    const int c = N / 2;
    const float da = live ? __ldg(&deapod[ix]) : 0.f, db = has_b ? __ldg(&deapod[ix + 1]) : 0.f;

    float2 v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int iy = (t + i * TF + c) & (L - 1);         // FFT position (iy - c) mod L
        v[i] = make_float2(0.f, 0.f);
        if (live && iy < N) {
            const float dy = __ldg(&deapod[iy]);
            const float *row = x + (size_t)iy * N + ix;
            v[i].x = __ldg(row) * da * dy;
            if (has_b) v[i].y = __ldg(row + 1) * db * dy;
        }
    }
    fft_reg<L, -1>(v, s, tw, t);
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 16; ++i) s[FFT_PAD(t + i * TF)] = v[i];
    __syncthreads();
    if (!live) return;
    // untangle: A[k] = (Z[k] + conj Z[-k])/2, B[k] = (Z[k] - conj Z[-k])/(2i), k = 0..L/2
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int k = t + i * TF;
        const float2 zk = v[i], zm = s[FFT_PAD((L - k) & (L - 1))];
        float2 *dst = T + (size_t)k * N + ix;
        dst[0] = make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
        if (has_b) dst[1] = make_float2(0.5f * (zk.y + zm.y), 0.5f * (zm.x - zk.x));
    }
    if (t == 0) {
        const float2 z = v[8];                              // k = L/2 is its own mirror
        float2 *dst = T + (size_t)(L / 2) * N + ix;
        dst[0] = make_float2(z.x, 0.f);
        if (has_b) dst[1] = make_float2(z.y, 0.f);
    }
}

// ---- second half of F2: rows ky = 0..L/2 of T -> centred grid rows ky and -ky ----------------
template <int L>
__global__ void __launch_bounds__(FftCfg<L>::THREADS)
rowpass_fwd_kernel(const float2 *__restrict__ T, float2 *__restrict__ grid,
                   const float2 *__restrict__ tw, int N, int mirror)
{
    extern __shared__ __align__(16) float2 s_fft[];
    using C = FftCfg<L>;
    constexpr int TF = C::TF;
    const int f = threadIdx.x / TF, t = threadIdx.x - f * TF;
    float2 *s = s_fft + f * C::PADLEN;
    const int ky = blockIdx.x * C::NF + f;
    const bool live = ky <= L / 2;
    const int c = N / 2;

    float2 v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int ix = (t + i * TF + c) & (L - 1);
        v[i] = (live && ix < N) ? __ldg(&T[(size_t)ky * N + ix]) : make_float2(0.f, 0.f);
    }
    fft_reg<L, -1>(v, s, tw, t);
    if (!live) return;
    const int cy = (ky + L / 2) & (L - 1);
    float2 *row = grid + (size_t)cy * L;
#pragma unroll
    for (int i = 0; i < 16; ++i) row[(t + i * TF + L / 2) & (L - 1)] = v[i];
    if (mirror && ky != 0 && ky != L / 2) {
        float2 *mrow = grid + (size_t)(L - cy) * L;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const int cx = (t + i * TF + L / 2) & (L - 1);
            mrow[(L - cx) & (L - 1)] = cconj(v[i]);
        }
    }
}

// ---- first half of A3: Hermitian part of grid rows ky = 0..L/2 -> T ---------------------------
template <int L>
__global__ void __launch_bounds__(FftCfg<L>::THREADS)
rowpass_inv_kernel(const float2 *__restrict__ grid, float2 *__restrict__ T,
                   const float2 *__restrict__ tw, int N, int fold)
{
    extern __shared__ __align__(16) float2 s_fft[];
    using C = FftCfg<L>;
    constexpr int TF = C::TF;
    const int f = threadIdx.x / TF, t = threadIdx.x - f * TF;
    float2 *s = s_fft + f * C::PADLEN;
    const int ky = blockIdx.x * C::NF + f;
    const bool live = ky <= L / 2;
    const int c = N / 2;
    const int cy = (ky + L / 2) & (L - 1);
    const float2 *row = grid + (size_t)cy * L, *mrow = grid + (size_t)((L - cy) & (L - 1)) * L;

    float2 v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int cx = (t + i * TF + L / 2) & (L - 1);
        v[i] = make_float2(0.f, 0.f);
        if (live) {
            v[i] = __ldg(&row[cx]);
            if (fold) {
                const float2 w = __ldg(&mrow[(L - cx) & (L - 1)]);
                v[i] = make_float2(0.5f * (v[i].x + w.x), 0.5f * (v[i].y - w.y));
            }
        }
    }
    fft_reg<L, +1>(v, s, tw, t);
    if (!live) return;
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int ix = (t + i * TF + c) & (L - 1);
        if (ix < N) T[(size_t)ky * N + ix] = v[i];
    }
}

// ---- second half of A3 + A4: column pairs of T -> image ---------------------------------------
template <int L>
__global__ void __launch_bounds__(FftCfg<L>::THREADS)
colpass_inv_kernel(const float2 *__restrict__ T, const float *__restrict__ deapod,
                   float *__restrict__ x, const float2 *__restrict__ tw, int N)
{
    extern __shared__ __align__(16) float2 s_fft[];
    using C = FftCfg<L>;
    constexpr int TF = C::TF;
    const int f = threadIdx.x / TF, t = threadIdx.x - f * TF;
    float2 *s = s_fft + f * C::PADLEN;
    const int p = blockIdx.x * C::NF + f, ix = 2 * p;
    const bool live = ix < N, has_b = ix + 1 < N;
    const int c = N / 2;

    float2 v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int k = t + i * TF;
        v[i] = make_float2(0.f, 0.f);
        if (live) {
            const bool up = k > L / 2;
            const float2 *src = T + (size_t)(up ? L - k : k) * N + ix;
            const float2 A = __ldg(src), B = has_b ? __ldg(src + 1) : make_float2(0.f, 0.f);
            if (k == 0 || k == L / 2) v[i] = make_float2(A.x, B.x);            // real by symmetry
            else if (!up) v[i] = make_float2(A.x - B.y, A.y + B.x);            // A + i B
            else v[i] = make_float2(A.x + B.y, B.x - A.y);                     // conj A + i conj B
        }
    }
    fft_reg<L, +1>(v, s, tw, t);
    if (!live) return;
    const float da = __ldg(&deapod[ix]), db = has_b ? __ldg(&deapod[ix + 1]) : 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int iy = (t + i * TF + c) & (L - 1);
        if (iy < N) {
            const float dy = __ldg(&deapod[iy]);
            float *row = x + (size_t)iy * N + ix;
            row[0] = v[i].x * da * dy;
            if (has_b) row[1] = v[i].y * db * dy;
        }
    }
}

// ---- dispatch on the FFT length -----------------------------------------------------------
bool fft_length_supported(int L) { return L >= 16 && L <= 8192 && (L & (L - 1)) == 0; }

template <int L>
static int fft2d_launch(int which, const DevicePlan &p, const void *in, void *out, int flag, cudaStream_t st)
{
    using C = FftCfg<L>;
    const int N = p.N;
    const int col_blocks = ((N + 1) / 2 + C::NF - 1) / C::NF, row_blocks = (L / 2 + 1 + C::NF - 1) / C::NF;
    const float2 *tw = p.tw_G;
    switch (which) {
    case 0:
        if (set_smem(colpass_fwd_kernel<L>, C::SMEM)) return -1;
        colpass_fwd_kernel<L><<<col_blocks, C::THREADS, C::SMEM, st>>>((const float *)in, p.deapod, (float2 *)out, tw, N);
        break;
    case 1:
        if (set_smem(rowpass_fwd_kernel<L>, C::SMEM)) return -1;
        rowpass_fwd_kernel<L><<<row_blocks, C::THREADS, C::SMEM, st>>>((const float2 *)in, (float2 *)out, tw, N, flag);
        break;
    case 2:
        if (set_smem(rowpass_inv_kernel<L>, C::SMEM)) return -1;
        rowpass_inv_kernel<L><<<row_blocks, C::THREADS, C::SMEM, st>>>((const float2 *)in, (float2 *)out, tw, N, flag);
        break;
    case 3:
        if (set_smem(colpass_inv_kernel<L>, C::SMEM)) return -1;
        colpass_inv_kernel<L><<<col_blocks, C::THREADS, C::SMEM, st>>>((const float2 *)in, p.deapod, (float *)out, tw, N);
        break;
    default:
        return -1;
    }
    count_launch();
    return 0;
}

int launch_fft2d_pass(int which, const DevicePlan &p, const void *in, void *out, int flag, cudaStream_t st)
{
    RADON_FOR_L(p.G, return fft2d_launch<LL>(which, p, in, out, flag, st);)
    return -1;
}

}  // namespace radon
