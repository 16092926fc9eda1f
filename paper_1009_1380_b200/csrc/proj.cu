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

// Sum NV values over the TF threads that share one FFT (thread t of FFT f in the CTA); every
// thread of the group gets the sum.  TF < 32: butterflies inside the group's lanes; otherwise
// butterflies inside each warp, then the group's warps through s_red in warp order (fixed
// order: bitwise reproducible).  All threads of the CTA must call it.
template <int TF, int NV>
__device__ __forceinline__ void group_sum(float (&v)[NV], float *s_red, int f)
{
    constexpr int WIDTH = TF < 32 ? TF : 32;
#pragma unroll
    for (int i = 0; i < NV; ++i)
#pragma unroll
        for (int o = WIDTH / 2; o > 0; o >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], o);
    if constexpr (TF > 32) {
        constexpr int WG = TF / 32;                       // warps per group
        const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
        __syncthreads();                                  // s_red free (a previous reduction was read)
        if (lane == 0)
#pragma unroll
            for (int i = 0; i < NV; ++i) s_red[warp * NV + i] = v[i];
        __syncthreads();
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            float a = 0.f;
            for (int w = 0; w < WG; ++w) a += s_red[(f * WG + w) * NV + i];
            v[i] = a;
        }
    }
}

// The polynomial sinogram filter along one projection held in registers (
// filter.cu has the stand-alone kernels): z[i] is element idx(i) = t + i*TF of the row (only
// elements < n count), q the orthonormal basis (n x FILTER_MAXQ floats, orders <= 3 in the first
// four columns).  NR rows at once (the pair kernels hold two projections per thread).
template <int TF, int NR>
__device__ __forceinline__ void filter_rows_in_registers(float (&z)[NR][16], const float *__restrict__ q, int n,
                                                         int t, int f, float *s_red)
{
    float c[NR * FILTER_FUSED_Q];
#pragma unroll
    for (int i = 0; i < NR * FILTER_FUSED_Q; ++i) c[i] = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int k = t + i * TF;
        if (k < n) {
            const float4 b = __ldg(reinterpret_cast<const float4 *>(q + (size_t)k * FILTER_MAXQ));
#pragma unroll
            for (int r = 0; r < NR; ++r) {
                c[r * 4 + 0] = fmaf(b.x, z[r][i], c[r * 4 + 0]); c[r * 4 + 1] = fmaf(b.y, z[r][i], c[r * 4 + 1]);
                c[r * 4 + 2] = fmaf(b.z, z[r][i], c[r * 4 + 2]); c[r * 4 + 3] = fmaf(b.w, z[r][i], c[r * 4 + 3]);
            }
        }
    }
    group_sum<TF, NR * FILTER_FUSED_Q>(c, s_red, f);
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int k = t + i * TF;
        if (k < n) {
            const float4 b = __ldg(reinterpret_cast<const float4 *>(q + (size_t)k * FILTER_MAXQ));
#pragma unroll
            for (int r = 0; r < NR; ++r) {
                float fit = b.x * c[r * 4 + 0];
                fit = fmaf(b.y, c[r * 4 + 1], fit); fit = fmaf(b.z, c[r * 4 + 2], fit); fit = fmaf(b.w, c[r * 4 + 3], fit);
                z[r][i] -= fit;
            }
        }
    }
}
constexpr int PROJ_RED_FLOATS = 32 * 2 * FILTER_FUSED_Q;     // up to 32 warps x 8 values

// BLUE: Bluestein form (two FFTs); false: n == L is a power of two, one FFT.
// FILT: the polynomial filter along the projection, on the output (INV, after `sub`) or the input.
template <int L, bool INV, bool BLUE, bool FILT>
__global__ void __launch_bounds__(ProjCfg<L>::THREADS, (BLUE || FILT) ? 1 : ProjCfg<L>::MIN_CTAS)
proj_kernel(const float *__restrict__ in, float *__restrict__ out,
            const float2 *__restrict__ ta, const float2 *__restrict__ tb,
            const float2 *__restrict__ hf, const float2 *__restrict__ tw, int n, int n_rows, int half,
            const float *__restrict__ dens, const float *__restrict__ sub, const float *__restrict__ q)
{
    extern __shared__ __align__(16) float2 s_fft[];
    __shared__ float s_red[FILT ? PROJ_RED_FLOATS : 1];
    pdl_prologue();
    using C = ProjCfg<L>;
    constexpr int TF = C::TF;
    const int f = threadIdx.x / TF, t = threadIdx.x - f * TF;
    float2 *s = s_fft + f * C::PADLEN;
    const int row = blockIdx.x * C::NF + f;
    const bool live = row < n_rows;

    float2 v[16];
    if constexpr (!INV && FILT) {
        float z[1][16];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const int sidx = t + i * TF;
            z[0][i] = (live && sidx < n) ? __ldg(&in[(size_t)row * n + sidx]) : 0.f;
        }
        filter_rows_in_registers<TF, 1>(z, q, n, t, f, s_red);
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const int sidx = t + i * TF;
            v[i] = make_float2(0.f, 0.f);
            if (live && sidx < n) { const float2 a = __ldg(&ta[sidx]); v[i] = make_float2(z[0][i] * a.x, z[0][i] * a.y); }
        }
    } else {
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
    }
    fft_reg<L, -1, true>(v, s, tw, t, f);          // the FFTs of a CTA only meet their own threads
    if constexpr (BLUE) {
#pragma unroll
        for (int i = 0; i < 16; ++i) v[i] = cmul(v[i], __ldg(&hf[t + i * TF]));
        fft_sync<TF, true>(f);
        fft_reg<L, +1, true>(v, s, tw, t, f);
    }
    pdl_trigger();
    if constexpr (INV) {
        float z[1][16];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const int k = t + i * TF;
            z[0][i] = (live && k < n) ? cmul(v[i], __ldg(&tb[k])).x : 0.f;
        }
        if (sub != nullptr) {                                      // residual Radon{x} - data (one branch: the loads stay batched)
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                const int k = t + i * TF;
                z[0][i] -= (live && k < n) ? __ldg(&sub[(size_t)row * n + k]) : 0.f;
            }
        }
        if constexpr (FILT) filter_rows_in_registers<TF, 1>(z, q, n, t, f, s_red);
        if (!live) return;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const int k = t + i * TF;
            if (k < n) out[(size_t)row * n + k] = z[0][i];
        }
    } else {
        if (!live) return;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const int k = t + i * TF;
            if (k < n) {
                float2 r = cmul(v[i], __ldg(&tb[k]));
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
template <int L, bool INV, bool FILT>
__global__ void __launch_bounds__(ProjCfg<L>::THREADS, FILT ? (ProjCfg<L>::MIN_CTAS > 1 ? ProjCfg<L>::MIN_CTAS / 2 : 1) : ProjCfg<L>::MIN_CTAS)
proj_pair_kernel(const float *__restrict__ in, float *__restrict__ out,
                 const float2 *__restrict__ ta, const float2 *__restrict__ tb,
                 const float2 *__restrict__ tw, int n_rows, const float *__restrict__ dens,
                 const float *__restrict__ sub, const float *__restrict__ q)
{
    extern __shared__ __align__(16) float2 s_fft[];
    __shared__ float s_red[FILT ? PROJ_RED_FLOATS : 1];
    pdl_prologue();
    using C = ProjCfg<L>;
    constexpr int TF = C::TF, n = L, c = L / 2;
    const int f = threadIdx.x / TF, t = threadIdx.x - f * TF;
    float2 *s = s_fft + f * C::PADLEN;
    const int r0 = 2 * (blockIdx.x * C::NF + f), r1 = r0 + 1;
    const bool live0 = r0 < n_rows, live1 = r1 < n_rows;

    float2 v[16];
    if constexpr (!INV && FILT) {
        float z[2][16];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const int sidx = t + i * TF;
            z[0][i] = live0 ? __ldg(&in[(size_t)r0 * n + sidx]) : 0.f;
            z[1][i] = live1 ? __ldg(&in[(size_t)r1 * n + sidx]) : 0.f;
        }
        filter_rows_in_registers<TF, 2>(z, q, n, t, f, s_red);
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const float a = __ldg(&ta[t + i * TF]).x;
            v[i] = make_float2(z[0][i] * a, z[1][i] * a);
        }
    } else {
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
    }
    fft_reg<L, -1, true>(v, s, tw, t, f);
    pdl_trigger();
    if (INV) {
        float z[2][16];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const float b = __ldg(&tb[t + i * TF]).x;
            z[0][i] = v[i].x * b;
            z[1][i] = -v[i].y * b;
        }
        if (sub != nullptr) {                                      // residual Radon{x} - data (one branch: the loads stay batched)
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                const int k = t + i * TF;
                z[0][i] -= live0 ? __ldg(&sub[(size_t)r0 * n + k]) : 0.f;
                z[1][i] -= live1 ? __ldg(&sub[(size_t)r1 * n + k]) : 0.f;
            }
        }
        if constexpr (FILT) filter_rows_in_registers<TF, 2>(z, q, n, t, f, s_red);
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const int k = t + i * TF;
            if (live0) out[(size_t)r0 * n + k] = z[0][i];
            if (live1) out[(size_t)r1 * n + k] = z[1][i];
        }
    } else {
        fft_sync<TF, true>(f);
#pragma unroll
        for (int i = 0; i < 16; ++i) s[FFT_PAD(t + i * TF)] = v[i];
        fft_sync<TF, true>(f);
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
static int proj_launch(bool inv, bool half, const DevicePlan &p, const float *in, float *out, const float *dens,
                       cudaStream_t st, const ProjExtra &ex)
{
    using C = ProjCfg<L>;
    const int blocks = (p.n_angles + C::NF - 1) / C::NF;
    const bool filt = ex.q != nullptr;
#define RADON_PROJ(INV_, BLUE_, FILT_)                                                                   \
    {                                                                                                    \
        if (set_smem(proj_kernel<L, INV_, BLUE_, FILT_>, C::SMEM)) return -1;                            \
        launch_pdl(p.pdl, proj_kernel<L, INV_, BLUE_, FILT_>, blocks, C::THREADS, C::SMEM, st,                  \
            in, out, p.chirp_a, p.chirp_b, p.chirp_hf, p.tw_P, p.n_det, p.n_angles, half ? 1 : 0, dens,  \
            ex.sub, ex.q);                                                                               \
    }
#define RADON_PROJ_PAIR(INV_, FILT_)                                                                     \
    {                                                                                                    \
        if (set_smem(proj_pair_kernel<L, INV_, FILT_>, C::SMEM)) return -1;                              \
        launch_pdl(p.pdl, proj_pair_kernel<L, INV_, FILT_>, pair_blocks, C::THREADS, C::SMEM, st,               \
            in, out, p.chirp_a, p.chirp_b, p.tw_P, p.n_angles, dens, ex.sub, ex.q);                      \
    }
    const bool blue = p.chirp_hf != nullptr;
    if (!blue && (!inv || half)) {        // n_det a power of two: two projections per FFT
        const int pair_blocks = ((p.n_angles + 1) / 2 + C::NF - 1) / C::NF;
        if (inv && filt) RADON_PROJ_PAIR(true, true)
        else if (inv) RADON_PROJ_PAIR(true, false)
        else if (filt) RADON_PROJ_PAIR(false, true)
        else RADON_PROJ_PAIR(false, false)
        count_launch();
        return 0;
    }
    if (inv && blue && filt) RADON_PROJ(true, true, true)
    else if (inv && blue) RADON_PROJ(true, true, false)
    else if (inv && filt) RADON_PROJ(true, false, true)
    else if (inv) RADON_PROJ(true, false, false)
    else if (blue && filt) RADON_PROJ(false, true, true)
    else if (blue) RADON_PROJ(false, true, false)
    else if (filt) RADON_PROJ(false, false, true)
    else RADON_PROJ(false, false, false)
#undef RADON_PROJ
#undef RADON_PROJ_PAIR
    count_launch();
    return 0;
}

int launch_proj(bool inv, bool half, const DevicePlan &p, const float *in, float *out, const float *dens, cudaStream_t st,
                const ProjExtra &ex)
{
    RADON_FOR_L(p.LP, return proj_launch<LL>(inv, half, p, in, out, dens, st, ex);)
    return -1;
}

}  // namespace radon
