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

#include <algorithm>
#include "fft_device.cuh"
#include "async_copy.cuh"

namespace radon {

template <int L>
struct FftCfg {
    static constexpr int TF = L / 16;                                  // threads per FFT
    static constexpr int NF = (TF >= 128) ? 1 : 128 / TF;              // FFTs per CTA
    static constexpr int THREADS = NF * TF;
    static constexpr int PADLEN = fft_padded_len(L);
    static constexpr size_t SMEM = (size_t)NF * PADLEN * sizeof(float2);
};

// Column passes: a CTA transforms NFC column PAIRS (2 NFC adjacent image columns).  All global
// traffic is cooperative, the pair index fastest across lanes, so that a warp touches 2 NFC
// adjacent floats of each image row / NFC adjacent (A, B) pairs of each T row -- whole 32-byte
// sectors -- instead of one sector per lane; the FFT threads pick their registers up from
// shared memory (ncu, round 1b: the per-lane version spent its time in the L1 sector stage,
// 31.5 sectors per store request, 4x write amplification into L2).
template <int L>
struct ColCfg {
    static constexpr int TF = L / 16;
#ifndef RADON_COL_NFC
#define RADON_COL_NFC 4
#endif
    static constexpr int NFC_WANT = (128 / TF > RADON_COL_NFC) ? 128 / TF : RADON_COL_NFC;
    static constexpr int NFC = (NFC_WANT * TF > 1024) ? 1024 / TF : NFC_WANT;   // column pairs per CTA
    static constexpr int THREADS = NFC * TF;
    static constexpr int SKEW = (16 / NFC > 1) ? 16 / NFC : 1;   // pairs start in distinct bank pairs
    static constexpr int STRIDE = fft_padded_len(L) + SKEW;
    static constexpr size_t SMEM = (size_t)NFC * STRIDE * sizeof(float2);
};

// ---- F1 + first half of F2 ------------------------------------------------------------------
// S2: sigma = 2 exactly (L == 2 N, N even).  Then element t + i TF of a zero-padded line is inside
// the image for i = 0..3 and 12..15 and exactly zero for i = 4..11, whatever t: the zero inputs of
// the first radix-16 pass (forward) and the unused outputs of the last one (inverse) are known at
// compile time and the butterflies that only move zeros / unused values are never generated.
template <int L, bool S2>
__global__ void __launch_bounds__(ColCfg<L>::THREADS)
colpass_fwd_kernel(const float *__restrict__ x, const float *__restrict__ deapod,
                   float2 *__restrict__ T, const float2 *__restrict__ tw, int N)
{
    extern __shared__ __align__(16) float2 s_fft[];
    pdl_prologue();
    using C = ColCfg<L>;
    constexpr int TF = C::TF, NFC = C::NFC;
    const int c = N / 2;
    const bool even = (N & 1) == 0;
    {   // cooperative load: thread -> (row iy, pair fc), fc fastest; de-apodise; FFT position (iy - c) mod L
        const int fc = threadIdx.x % NFC, ix = 2 * (blockIdx.x * NFC + fc);
        float2 *sf = s_fft + fc * C::STRIDE;
        if (ix < N) {
            const bool has_b = ix + 1 < N;
            const float da = __ldg(&deapod[ix]), db = has_b ? __ldg(&deapod[ix + 1]) : 0.f;
            // batches of 8 rows: all loads of a batch are in flight before the first is used
            constexpr int RS = C::THREADS / NFC;
            for (int iy0 = threadIdx.x / NFC; iy0 < N; iy0 += 8 * RS) {
                float2 v[8];
                float dy[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    const int iy = iy0 + q * RS;
                    v[q] = make_float2(0.f, 0.f);
                    dy[q] = 0.f;
                    if (iy < N) {
                        dy[q] = __ldg(&deapod[iy]);
                        const float *row = x + (size_t)iy * N + ix;
                        if (even) v[q] = __ldg(reinterpret_cast<const float2 *>(row));
                        else { v[q].x = __ldg(row); v[q].y = has_b ? __ldg(row + 1) : 0.f; }
                    }
                }
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    const int iy = iy0 + q * RS;
                    if (iy < N) sf[FFT_PAD((iy - c) & (L - 1))] = make_float2(v[q].x * da * dy[q], v[q].y * db * dy[q]);
                }
            }
        }
    }
    __syncthreads();
    const int f = threadIdx.x / TF, t = threadIdx.x - f * TF;
    float2 *s = s_fft + f * C::STRIDE;
    const bool live = 2 * (blockIdx.x * NFC + f) < N;
    float2 v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int iy = (t + i * TF + c) & (L - 1);         // zero padding pruned: rows >= N were never staged
        if (S2) v[i] = (i < 4 || i >= 12) ? (live ? s[FFT_PAD(t + i * TF)] : make_float2(0.f, 0.f)) : make_float2(0.f, 0.f);
        else v[i] = (live && iy < N) ? s[FFT_PAD(t + i * TF)] : make_float2(0.f, 0.f);
    }
    // from here to the cooperative store the four FFTs of the CTA only meet their own threads
    fft_sync<TF, true>(f);
    fft_reg<L, -1, true>(v, s, tw, t, f);
    fft_sync<TF, true>(f);
#pragma unroll
    for (int i = 0; i < 16; ++i) s[FFT_PAD(t + i * TF)] = v[i];
    pdl_trigger();
    __syncthreads();
    {   // cooperative store: thread -> (ky, pair fc); untangle the packed pair:
        // A[k] = (Z[k] + conj Z[-k])/2, B[k] = (Z[k] - conj Z[-k])/(2i), k = 0..L/2
        const int fc = threadIdx.x % NFC, ix = 2 * (blockIdx.x * NFC + fc);
        const float2 *sf = s_fft + fc * C::STRIDE;
        if (ix < N) {
            const bool has_b = ix + 1 < N;
            for (int k = threadIdx.x / NFC; k <= L / 2; k += C::THREADS / NFC) {
                const float2 zk = sf[FFT_PAD(k)], zm = sf[FFT_PAD((L - k) & (L - 1))];
                const float2 A = make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
                const float2 B = make_float2(0.5f * (zk.y + zm.y), 0.5f * (zm.x - zk.x));
                float2 *dst = T + (size_t)k * N + ix;
                if (even) *reinterpret_cast<float4 *>(dst) = make_float4(A.x, A.y, B.x, B.y);
                else { dst[0] = A; if (has_b) dst[1] = B; }
            }
        }
    }
}

// ---- second half of F2: rows ky = 0..L/2 of T -> centred grid rows ky and -ky ----------------
template <int L, bool S2>
__global__ void __launch_bounds__(FftCfg<L>::THREADS, (FftCfg<L>::THREADS <= 256) ? 1024 / FftCfg<L>::THREADS : 1)   // 64 registers: four CTAs of 256
rowpass_fwd_kernel(const float2 *__restrict__ T, float2 *__restrict__ grid,
                   const float2 *__restrict__ tw, int N, int mirror, int KW)
{
    extern __shared__ __align__(16) float2 s_fft[];
    pdl_prologue();
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
        if (S2) v[i] = (i < 4 || i >= 12) ? (live ? __ldg(&T[(size_t)ky * N + ix]) : make_float2(0.f, 0.f)) : make_float2(0.f, 0.f);
        else v[i] = (live && ix < N) ? __ldg(&T[(size_t)ky * N + ix]) : make_float2(0.f, 0.f);
    }
    fft_reg<L, -1, true>(v, s, tw, t, f);
    pdl_trigger();
    if (!live) return;
    const int cy = (ky + L / 2) & (L - 1);
    float2 *row = grid + (size_t)cy * L;
#pragma unroll
    for (int i = 0; i < 16; ++i) row[(t + i * TF + L / 2) & (L - 1)] = v[i];
    // mirror == 1: every row -ky; mirror == 2: only the rows the Hermitian-half gather reads
    // besides ky = 0 .. L/2, i.e. -KW/2 <= ky' < 0 and L/2 < ky' <= L/2 + KW/2 - 1 (mod L)
    const bool want = mirror == 1 || (mirror == 2 && (ky <= KW / 2 || ky >= L / 2 - (KW / 2 - 1)));
    if (want && ky != 0 && ky != L / 2) {
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
    pdl_prologue();
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
    fft_reg<L, +1, true>(v, s, tw, t, f);
    pdl_trigger();
    if (!live) return;
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int ix = (t + i * TF + c) & (L - 1);
        if (ix < N) T[(size_t)ky * N + ix] = v[i];
    }
}

// ---- first half of A3, Hermitian-half form: grid rows ky = 0..L/2 as they are -> T ------------
// Persistent CTAs; the copy engine fetches the NEXT group of rows (one bulk copy per row)
// into a staging buffer while the warps transform the current one, so the DRAM latency of
// the row reads is off the critical path (ncu, round 1b: the per-thread-load version issued
// on 32 % of cycles, waiting on its 16 loads per thread).
template <int L>
struct RowStageCfg {
    using C = FftCfg<L>;
    static constexpr size_t STAGE_BYTES = (size_t)C::NF * L * sizeof(float2);
    static constexpr size_t SMEM = C::SMEM + STAGE_BYTES;
};

template <int L, bool S2>
__global__ void __launch_bounds__(FftCfg<L>::THREADS, (FftCfg<L>::THREADS <= 256) ? 3 : 1)
rowpass_inv_staged_kernel(const float2 *__restrict__ grid, float2 *__restrict__ T,
                          const float2 *__restrict__ tw, int N, int n_groups)
{
    extern __shared__ __align__(128) float2 s_rows[];   // FFT scratch, then the staged rows
    pdl_prologue();
    using C = FftCfg<L>;
    constexpr int TF = C::TF, NF = C::NF;
    __shared__ __align__(8) uint64_t bar;
    float2 *stage = s_rows + NF * C::PADLEN;                 // NF rows of L, 16-byte aligned
    const int f = threadIdx.x / TF, t = threadIdx.x - f * TF;
    float2 *s = s_rows + f * C::PADLEN;
    const int c = N / 2;

    auto fetch = [&](int g) {                               // one thread: rows of group g -> stage
        int n_live = 0;
        for (int q = 0; q < NF; ++q) n_live += (g * NF + q <= L / 2) ? 1 : 0;
        mbar_expect_tx(&bar, (uint32_t)(n_live * L * sizeof(float2)));
        for (int q = 0; q < NF; ++q) {
            const int ky = g * NF + q;
            if (ky > L / 2) break;
            const int cy = (ky + L / 2) & (L - 1);
            bulk_g2s(stage + q * L, grid + (size_t)cy * L, (uint32_t)(L * sizeof(float2)), &bar);
        }
    };
    if (threadIdx.x == 0) {
        mbar_init(&bar, 1);
        if ((int)blockIdx.x < n_groups) fetch(blockIdx.x);
    }
    __syncthreads();
    uint32_t parity = 0;
    for (int g = blockIdx.x; g < n_groups; g += gridDim.x) {
        const int ky = g * NF + f;
        const bool live = ky <= L / 2;
        mbar_wait(&bar, parity);
        parity ^= 1u;
        float2 v[16];
#pragma unroll
        for (int i = 0; i < 16; ++i)
            v[i] = live ? stage[f * L + ((t + i * TF + L / 2) & (L - 1))] : make_float2(0.f, 0.f);
        // The staging buffer is read through the generic proxy and refilled through the async
        // proxy: without this fence the refill can overtake reads still in flight (observed:
        // run-to-run differences of 2 % in the adjoint).
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();                                    // stage is free; s is free (previous FFT done)
        if (threadIdx.x == 0 && g + (int)gridDim.x < n_groups) fetch(g + gridDim.x);
        if (g + (int)gridDim.x >= n_groups) pdl_trigger();      // this CTA's last group
        fft_reg<L, +1, true>(v, s, tw, t, f);
        if (live) {
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                const int ix = (t + i * TF + c) & (L - 1);
                if (S2) { if (i < 4 || i >= 12) T[(size_t)ky * N + ix] = v[i]; }
                else if (ix < N) T[(size_t)ky * N + ix] = v[i];
            }
        }
    }
}

// ---- second half of A3 + A4: column pairs of T -> image ---------------------------------------
template <int L, bool S2>
__global__ void __launch_bounds__(ColCfg<L>::THREADS)
colpass_inv_kernel(const float2 *__restrict__ T, const float *__restrict__ deapod,
                   float *x, const float2 *__restrict__ tw, int N, int update, float alpha, float tau)
{
    extern __shared__ __align__(16) float2 s_fft[];
    pdl_prologue();
    using C = ColCfg<L>;
    constexpr int TF = C::TF, NFC = C::NFC;
    const int c = N / 2;
    const bool even = (N & 1) == 0;
    const int fc = threadIdx.x % NFC, ixc = 2 * (blockIdx.x * NFC + fc);
    float2 *sf = s_fft + fc * C::STRIDE;
    if (ixc < N) {   // cooperative load: thread -> (ky, pair fc); pack Z = A + i B, Z[-k] = conj A + i conj B
        const bool has_b = ixc + 1 < N;
        constexpr int RS = C::THREADS / NFC;
        for (int k0 = threadIdx.x / NFC; k0 <= L / 2; k0 += 8 * RS) {
            float2 A[8], B[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) {       // 8 loads in flight
                const int k = k0 + q * RS;
                A[q] = B[q] = make_float2(0.f, 0.f);
                if (k <= L / 2) {
                    const float2 *src = T + (size_t)k * N + ixc;
                    if (even) { const float4 w = __ldg(reinterpret_cast<const float4 *>(src)); A[q] = make_float2(w.x, w.y); B[q] = make_float2(w.z, w.w); }
                    else { A[q] = __ldg(src); if (has_b) B[q] = __ldg(src + 1); }
                }
            }
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const int k = k0 + q * RS;
                if (k > L / 2) continue;
                if (k == 0 || k == L / 2) sf[FFT_PAD(k)] = make_float2(A[q].x, B[q].x);        // real by symmetry
                else {
                    sf[FFT_PAD(k)] = make_float2(A[q].x - B[q].y, A[q].y + B[q].x);
                    sf[FFT_PAD(L - k)] = make_float2(A[q].x + B[q].y, B[q].x - A[q].y);
                }
            }
        }
    }
    __syncthreads();
    const int f = threadIdx.x / TF, t = threadIdx.x - f * TF;
    float2 *s = s_fft + f * C::STRIDE;
    const bool live = 2 * (blockIdx.x * NFC + f) < N;
    float2 v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = live ? s[FFT_PAD(t + i * TF)] : make_float2(0.f, 0.f);
    fft_sync<TF, true>(f);
    fft_reg<L, +1, true>(v, s, tw, t, f);
    fft_sync<TF, true>(f);
#pragma unroll
    for (int i = 0; i < 16; ++i)
        if (!S2 || i < 4 || i >= 12) s[FFT_PAD(t + i * TF)] = v[i];       // S2: the other rows are cropped
    pdl_trigger();
    __syncthreads();
    if (ixc < N) {   // cooperative store: thread -> (row iy, pair fc); crop, de-apodise
        const bool has_b = ixc + 1 < N;
        const float da = __ldg(&deapod[ixc]), db = has_b ? __ldg(&deapod[ixc + 1]) : 0.f;
        for (int iy = threadIdx.x / NFC; iy < N; iy += C::THREADS / NFC) {
            const float dy = __ldg(&deapod[iy]);
            const float2 z = sf[FFT_PAD((iy - c) & (L - 1))];
            float *row = x + (size_t)iy * N + ixc;
            float ga = z.x * da * dy, gb = z.y * db * dy;
            if (update) {
                // solver iteration: x <- S_tau(x - alpha g), g = Radon^T{residual}
                // just computed; the thread that writes a pixel is the one that reads it
                float xa, xb = 0.f;
                if (even) { const float2 xo = *reinterpret_cast<const float2 *>(row); xa = xo.x; xb = xo.y; }
                else { xa = row[0]; if (has_b) xb = row[1]; }
                const float va = fmaf(-alpha, ga, xa), vb = fmaf(-alpha, gb, xb);
                ga = copysignf(fmaxf(fabsf(va) - tau, 0.f), va);
                gb = copysignf(fmaxf(fabsf(vb) - tau, 0.f), vb);
            }
            if (even) *reinterpret_cast<float2 *>(row) = make_float2(ga, gb);
            else { row[0] = ga; if (has_b) row[1] = gb; }
        }
    }
}

// ---- dispatch on the FFT length -----------------------------------------------------------
bool fft_length_supported(int L)
{
    if (L >= 16 && L <= 8192 && (L & (L - 1)) == 0) return true;
    return fft_composite_split(L, nullptr, nullptr);
}

template <int L>
static int fft2d_launch(int which, const DevicePlan &p, const void *in, void *out, int flag, cudaStream_t st,
                        const IstaUpdate *upd)
{
    using C = FftCfg<L>;
    using CC = ColCfg<L>;
    const int N = p.N;
    const int col_blocks = ((N + 1) / 2 + CC::NFC - 1) / CC::NFC, row_blocks = (L / 2 + 1 + C::NF - 1) / C::NF;
    const float2 *tw = p.tw_G;
    const bool s2 = (L == 2 * N) && (N % 2 == 0) && L >= 64;      // sigma = 2: pruned first / last radix-16 pass
    switch (which) {
    case 0:
        if (s2) {
            if (set_smem(colpass_fwd_kernel<L, true>, CC::SMEM)) return -1;
            launch_pdl(p.pdl, colpass_fwd_kernel<L, true>, col_blocks, CC::THREADS, CC::SMEM, st, (const float *)in, p.deapod, (float2 *)out, tw, N);
        } else {
            if (set_smem(colpass_fwd_kernel<L, false>, CC::SMEM)) return -1;
            launch_pdl(p.pdl, colpass_fwd_kernel<L, false>, col_blocks, CC::THREADS, CC::SMEM, st, (const float *)in, p.deapod, (float2 *)out, tw, N);
        }
        break;
    case 1:
        if (s2) {
            if (set_smem(rowpass_fwd_kernel<L, true>, C::SMEM)) return -1;
            launch_pdl(p.pdl, rowpass_fwd_kernel<L, true>, row_blocks, C::THREADS, C::SMEM, st, (const float2 *)in, (float2 *)out, tw, N, flag, p.W);
        } else {
            if (set_smem(rowpass_fwd_kernel<L, false>, C::SMEM)) return -1;
            launch_pdl(p.pdl, rowpass_fwd_kernel<L, false>, row_blocks, C::THREADS, C::SMEM, st, (const float2 *)in, (float2 *)out, tw, N, flag, p.W);
        }
        break;
    case 2:
        if (flag) {
            if (set_smem(rowpass_inv_kernel<L>, C::SMEM)) return -1;
            launch_pdl(p.pdl, rowpass_inv_kernel<L>, row_blocks, C::THREADS, C::SMEM, st, (const float2 *)in, (float2 *)out, tw, N, flag);
        } else {
            using RS = RowStageCfg<L>;
            const int per_sm = std::max(1, std::min(8, (int)((220u << 10) / (RS::SMEM + 1024))));
            const int ctas = std::min(row_blocks, p.n_sm * per_sm);
            if (s2) {
                if (set_smem(rowpass_inv_staged_kernel<L, true>, RS::SMEM)) return -1;
                launch_pdl(p.pdl, rowpass_inv_staged_kernel<L, true>, ctas, C::THREADS, RS::SMEM, st, (const float2 *)in, (float2 *)out, tw, N, row_blocks);
            } else {
                if (set_smem(rowpass_inv_staged_kernel<L, false>, RS::SMEM)) return -1;
                launch_pdl(p.pdl, rowpass_inv_staged_kernel<L, false>, ctas, C::THREADS, RS::SMEM, st, (const float2 *)in, (float2 *)out, tw, N, row_blocks);
            }
        }
        break;
    case 3:
        if (s2) {
            if (set_smem(colpass_inv_kernel<L, true>, CC::SMEM)) return -1;
            launch_pdl(p.pdl, colpass_inv_kernel<L, true>, col_blocks, CC::THREADS, CC::SMEM, st, (const float2 *)in, p.deapod, (float *)out, tw, N,
                                                                                     upd ? 1 : 0, upd ? upd->alpha : 0.f, upd ? upd->tau : 0.f);
        } else {
            if (set_smem(colpass_inv_kernel<L, false>, CC::SMEM)) return -1;
            launch_pdl(p.pdl, colpass_inv_kernel<L, false>, col_blocks, CC::THREADS, CC::SMEM, st, (const float2 *)in, p.deapod, (float *)out, tw, N,
                                                                                      upd ? 1 : 0, upd ? upd->alpha : 0.f, upd ? upd->tau : 0.f);
        }
        break;
    default:
        return -1;
    }
    count_launch();
    return 0;
}

int launch_fft2d_pass(int which, const DevicePlan &p, const void *in, void *out, int flag, cudaStream_t st,
                      const IstaUpdate *upd)
{
    if ((p.G & (p.G - 1)) != 0) return launch_fft2d_composite(which, p, in, out, flag, st, upd);
    RADON_FOR_L(p.G, return fft2d_launch<LL>(which, p, in, out, flag, st, upd);)
    return -1;
}

}  // namespace radon
