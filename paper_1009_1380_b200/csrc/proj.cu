// proj.cu -- F4 / A1: the 1-D transforms along the projections ("1D inverse
// Fourier transforms are applied to interpolated points along the same radial lines").
//
// Centred DFT of length n = n_det along each projection,
//   Z[k] = (1/n) sum_s z[s] exp(-i 2 pi (k-c)(s-c)/n), c = n/2,
// as  b[k] * FFT_n(a .* z)[k]  when n is a power of two, else (any n) by Bluestein:
// b[k] * IFFT_L( FFT_L(a .* z) .* hf )[k] with L >= 2n-1 a power of two.  The two FFTs of the
// Bluestein form run back to back in registers (the output layout of fft_reg is its input
// layout), so the spectrum product costs no shared-memory round trip.
//   INV = false (A1): z = sinogram row (real), output Z (complex).
//   INV = true  (F4): z = conj(P), output Re Z, i.e. S = Re{(1/n) sum_k P exp(+i 2 pi j t/n)}.
#include "kernels.h"
#include "fft_device.cuh"

namespace radon {

template <int L>
struct ProjCfg {
    static constexpr int TF = L / 16;
    static constexpr int NF = (TF >= 128) ? 1 : 128 / TF;
    static constexpr int THREADS = NF * TF;
    static constexpr int PADLEN = fft_padded_len(L);
    static constexpr size_t SMEM = (size_t)NF * PADLEN * sizeof(float2);
    static constexpr int MIN_CTAS = 1024 / THREADS;      // <= 64 registers per thread
};

// BLUE: Bluestein form (two FFTs); false: n == L is a power of two, one FFT.
template <int L, bool INV, bool BLUE>
__global__ void __launch_bounds__(ProjCfg<L>::THREADS, BLUE ? 1 : ProjCfg<L>::MIN_CTAS)
proj_kernel(const float *__restrict__ in, float *__restrict__ out,
            const float2 *__restrict__ ta, const float2 *__restrict__ tb,
            const float2 *__restrict__ hf, const float2 *__restrict__ tw, int n, int n_rows, int half,
            const float *__restrict__ dens)
{
    extern __shared__ __align__(16) float2 s_fft[];
    using C = ProjCfg<L>;
    constexpr int TF = C::TF;
    const int f = threadIdx.x / TF, t = threadIdx.x - f * TF;
    float2 *s = s_fft + f * C::PADLEN;
    const int row = blockIdx.x * C::NF + f;
    const bool live = row < n_rows;

    float2 v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int sidx = t + i * TF;
        v[i] = make_float2(0.f, 0.f);
        if (live && sidx < n) {
            const float2 a = __ldg(&ta[sidx]);
            if (INV) {
                // half: the row holds k >= n/2 (and k = 0 for even n); P[c - j] = conj P[c + j]
                const int c = n >> 1;
                const bool mir = half && sidx < c && !(sidx == 0 && (n & 1) == 0);
                float2 p = __ldg(&reinterpret_cast<const float2 *>(in)[(size_t)row * n + (mir ? 2 * c - sidx : sidx)]);
                if (mir) p.y = -p.y;
                v[i] = make_float2(p.x * a.x + p.y * a.y, p.x * a.y - p.y * a.x);   // conj(p) * a
            } else {
                const float y = __ldg(&in[(size_t)row * n + sidx]);
                v[i] = make_float2(y * a.x, y * a.y);
            }
        }
    }
    fft_reg<L, -1>(v, s, tw, t);
    if constexpr (BLUE) {
#pragma unroll
        for (int i = 0; i < 16; ++i) v[i] = cmul(v[i], __ldg(&hf[t + i * TF]));
        __syncthreads();
        fft_reg<L, +1>(v, s, tw, t);
    }
    if (!live) return;
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int k = t + i * TF;
        if (k < n) {
            float2 r = cmul(v[i], __ldg(&tb[k]));
            if (INV) out[(size_t)row * n + k] = r.x;
            else {
                // radon_inverse: density compensation D applied to the sample
                if (dens != nullptr) { const float w = __ldg(&dens[(size_t)row * n + k]); r.x *= w; r.y *= w; }
                reinterpret_cast<float2 *>(out)[(size_t)row * n + k] = r;
            }
        }
    }
}

template <int L>
static int proj_launch(bool inv, bool half, const DevicePlan &p, const float *in, float *out, const float *dens, cudaStream_t st)
{
    using C = ProjCfg<L>;
    const int blocks = (p.n_angles + C::NF - 1) / C::NF;
#define RADON_PROJ(INV_, BLUE_)                                                                          \
    {                                                                                                    \
        if (set_smem(proj_kernel<L, INV_, BLUE_>, C::SMEM)) return -1;                                   \
        proj_kernel<L, INV_, BLUE_><<<blocks, C::THREADS, C::SMEM, st>>>(                                \
            in, out, p.chirp_a, p.chirp_b, p.chirp_hf, p.tw_P, p.n_det, p.n_angles, half ? 1 : 0, dens); \
    }
    const bool blue = p.chirp_hf != nullptr;
    if (inv && blue) RADON_PROJ(true, true)
    else if (inv) RADON_PROJ(true, false)
    else if (blue) RADON_PROJ(false, true)
    else RADON_PROJ(false, false)
#undef RADON_PROJ
    count_launch();
    return 0;
}

int launch_proj(bool inv, bool half, const DevicePlan &p, const float *in, float *out, const float *dens, cudaStream_t st)
{
    RADON_FOR_L(p.LP, return proj_launch<LL>(inv, half, p, in, out, dens, st);)
    return -1;
}

}  // namespace radon
