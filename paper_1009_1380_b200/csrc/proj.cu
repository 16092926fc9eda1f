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

// ---- n_det a power of two: two projections per FFT ---------------------------------------------
// For n = L a power of two the centring phases are real (a[s] = (-1)^s, b[k] = (-1)^k / n), so
// real <-> Hermitian symmetry halves the work exactly as in the column passes of the 2-D FFT:
//   A1 (INV = false): rows y0, y1 real -> one FFT of a .* (y0 + i y1) = W; the two spectra are
//       untangled through shared memory, Y0[k] = b[k] (W[k] + conj W[-k])/2,
//       Y1[k] = b[k] (W[k] - conj W[-k])/(2i).
//   F4 (INV = true, Hermitian-half rows only): P0, P1 completed to Hermitian rows (the stored
//       half, mirrored and conjugated; the self-mirrored k = n/2 and the unpaired k = 0 keep
//       their real part: that is what Re{.} of the single-row form leaves of them), one FFT of
//       conj(P0 + i P1) .* a, r = b .* result; S0 = r.x, S1 = -r.y.
template <int L, bool INV>
__global__ void __launch_bounds__(ProjCfg<L>::THREADS, ProjCfg<L>::MIN_CTAS)
proj_pair_kernel(const float *__restrict__ in, float *__restrict__ out,
                 const float2 *__restrict__ ta, const float2 *__restrict__ tb,
                 const float2 *__restrict__ tw, int n_rows, const float *__restrict__ dens)
{
    extern __shared__ __align__(16) float2 s_fft[];
    using C = ProjCfg<L>;
    constexpr int TF = C::TF, n = L, c = L / 2;
    const int f = threadIdx.x / TF, t = threadIdx.x - f * TF;
    float2 *s = s_fft + f * C::PADLEN;
    const int r0 = 2 * (blockIdx.x * C::NF + f), r1 = r0 + 1;
    const bool live0 = r0 < n_rows, live1 = r1 < n_rows;

    float2 v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int sidx = t + i * TF;
        const float a = __ldg(&ta[sidx]).x;
        if (INV) {
            const bool self = sidx == 0 || sidx == c;            // keep the real part only
            const bool mir = sidx < c && sidx != 0;
            const int src = mir ? 2 * c - sidx : sidx;
            const float2 *P = reinterpret_cast<const float2 *>(in);
            float2 p0 = live0 ? __ldg(&P[(size_t)r0 * n + src]) : make_float2(0.f, 0.f);
            float2 p1 = live1 ? __ldg(&P[(size_t)r1 * n + src]) : make_float2(0.f, 0.f);
            if (mir) { p0.y = -p0.y; p1.y = -p1.y; }
            if (self) { p0.y = 0.f; p1.y = 0.f; }
            // z = p0 + i p1; v = conj(z) * a
            v[i] = make_float2((p0.x - p1.y) * a, -(p0.y + p1.x) * a);
        } else {
            const float y0 = live0 ? __ldg(&in[(size_t)r0 * n + sidx]) : 0.f;
            const float y1 = live1 ? __ldg(&in[(size_t)r1 * n + sidx]) : 0.f;
            v[i] = make_float2(y0 * a, y1 * a);
        }
    }
    fft_reg<L, -1>(v, s, tw, t);
    if (INV) {
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const int k = t + i * TF;
            const float b = __ldg(&tb[k]).x;
            if (live0) out[(size_t)r0 * n + k] = v[i].x * b;
            if (live1) out[(size_t)r1 * n + k] = -v[i].y * b;
        }
    } else {
        __syncthreads();
#pragma unroll
        for (int i = 0; i < 16; ++i) s[FFT_PAD(t + i * TF)] = v[i];
        __syncthreads();
        float2 *Y = reinterpret_cast<float2 *>(out);
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const int k = t + i * TF;
            const float2 wk = v[i], wm = s[FFT_PAD((L - k) & (L - 1))];
            const float b = __ldg(&tb[k]).x;
            float2 y0 = make_float2(0.5f * b * (wk.x + wm.x), 0.5f * b * (wk.y - wm.y));
            float2 y1 = make_float2(0.5f * b * (wk.y + wm.y), 0.5f * b * (wm.x - wk.x));
            if (dens != nullptr) {        // radon_inverse: density compensation
                if (live0) { const float w = __ldg(&dens[(size_t)r0 * n + k]); y0.x *= w; y0.y *= w; }
                if (live1) { const float w = __ldg(&dens[(size_t)r1 * n + k]); y1.x *= w; y1.y *= w; }
            }
            if (live0) Y[(size_t)r0 * n + k] = y0;
            if (live1) Y[(size_t)r1 * n + k] = y1;
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
    if (!blue && (!inv || half)) {        // n_det a power of two: two projections per FFT
        const int pair_blocks = ((p.n_angles + 1) / 2 + C::NF - 1) / C::NF;
        if (inv) {
            if (set_smem(proj_pair_kernel<L, true>, C::SMEM)) return -1;
            proj_pair_kernel<L, true><<<pair_blocks, C::THREADS, C::SMEM, st>>>(in, out, p.chirp_a, p.chirp_b, p.tw_P, p.n_angles, dens);
        } else {
            if (set_smem(proj_pair_kernel<L, false>, C::SMEM)) return -1;
            proj_pair_kernel<L, false><<<pair_blocks, C::THREADS, C::SMEM, st>>>(in, out, p.chirp_a, p.chirp_b, p.tw_P, p.n_angles, dens);
        }
        count_launch();
        return 0;
    }
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
