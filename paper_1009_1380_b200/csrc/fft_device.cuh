// fft_device.cuh -- register/shared-memory Stockham FFT for power-of-two lengths 16 .. 8192.
//
// No cuFFT (BASELINE.json north_star: "shared-memory radix 2D FFT of the oversampled image
// and batched 1D FFTs along each projection").  One FFT of length L is computed by
// TF = L/16 threads, 16 complex values per thread:
//   * input and output live in REGISTERS: thread t holds x[t + i*TF], i = 0..15, on entry and
//     X[t + i*TF] on exit (both coalesced across t when moved to or from global memory), so
//     the first pass needs no shared-memory fill and the last one no read-out;
//   * between passes the data cross shared memory once (write, barrier, read), skewed by one
//     element per 16 (FFT_PAD) so that every 64-bit access of a half-warp is conflict free;
//   * passes are radix 16 (two radix-4 layers in registers), preceded by one radix-2/4/8 pass
//     when log2 L is not a multiple of 4;
//   * the 15 twiddles of a radix-16 butterfly come from FOUR table loads (w^1, w^2, w^4, w^8;
//     table derived in fp64 at plan time) and 11 complex products, instead of 15 scattered
//     loads that would share the load/store pipe with the shared-memory traffic.
#pragma once
#include <cuda_runtime.h>

namespace radon {

#define FFT_PAD(i) ((i) + ((i) >> 4))
__host__ __device__ constexpr int fft_padded_len(int L) { return L + (L >> 4); }
__host__ __device__ constexpr int ilog2_c(int v) { return v <= 1 ? 0 : 1 + ilog2_c(v >> 1); }

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b)
{
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 cconj(float2 a) { return make_float2(a.x, -a.y); }
// a * w (SIGN < 0, forward) or a * conj(w) (SIGN > 0, inverse); w = exp(-i phi)
template <int SIGN>
__device__ __forceinline__ float2 cmul_tw(float2 a, float2 w)
{
    if (SIGN < 0) return make_float2(fmaf(a.x, w.x, -a.y * w.y), fmaf(a.x, w.y, a.y * w.x));
    return make_float2(fmaf(a.x, w.x, a.y * w.y), fmaf(-a.x, w.y, a.y * w.x));
}

// a * exp(SIGN * 2 pi i M / 16), M = 0..15, constants folded, trivial cases free
template <int M, int SIGN>
__device__ __forceinline__ float2 mul_w16(float2 a)
{
    constexpr float C1 = 0.92387953251128674f, S1 = 0.38268343236508977f, RH = 0.70710678118654752f;
    constexpr int m = M & 15;
    if constexpr (m == 0) return a;
    else if constexpr (m == 8) return make_float2(-a.x, -a.y);
    else if constexpr (m == 4) return SIGN < 0 ? make_float2(a.y, -a.x) : make_float2(-a.y, a.x);
    else if constexpr (m == 12) return SIGN < 0 ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
    else if constexpr (m == 2) return SIGN < 0 ? make_float2(RH * (a.x + a.y), RH * (a.y - a.x))
                                               : make_float2(RH * (a.x - a.y), RH * (a.y + a.x));
    else if constexpr (m == 6) return SIGN < 0 ? make_float2(RH * (a.y - a.x), -RH * (a.x + a.y))
                                               : make_float2(-RH * (a.x + a.y), RH * (a.x - a.y));
    else {
        // general: w = (cos(2 pi m/16), SIGN * sin(2 pi m/16))
        constexpr float cs[16] = {1.f, C1, RH, S1, 0.f, -S1, -RH, -C1, -1.f, -C1, -RH, -S1, 0.f, S1, RH, C1};
        constexpr float sn[16] = {0.f, S1, RH, C1, 1.f, C1, RH, S1, 0.f, -S1, -RH, -C1, -1.f, -C1, -RH, -S1};
        constexpr float wr = cs[m], wi = (SIGN < 0 ? -sn[m] : sn[m]);
        return make_float2(fmaf(a.x, wr, -a.y * wi), fmaf(a.x, wi, a.y * wr));
    }
}

template <int SIGN>
__device__ __forceinline__ void dft4(float2 &a, float2 &b, float2 &c, float2 &d)
{
    const float2 t0 = cadd(a, c), t1 = csub(a, c), t2 = cadd(b, d), t3 = csub(b, d);
    a = cadd(t0, t2);
    c = csub(t0, t2);
    if (SIGN < 0) {   // t1 -/+ i t3
        b = make_float2(t1.x + t3.y, t1.y - t3.x);
        d = make_float2(t1.x - t3.y, t1.y + t3.x);
    } else {
        b = make_float2(t1.x - t3.y, t1.y + t3.x);
        d = make_float2(t1.x + t3.y, t1.y - t3.x);
    }
}

// In-register DFT of R points (R = 2, 4, 8, 16), natural order in and out.
template <int R, int SIGN>
__device__ __forceinline__ void dft_reg(float2 (&v)[R])
{
    if constexpr (R == 2) {
        const float2 a = v[0], b = v[1];
        v[0] = cadd(a, b);
        v[1] = csub(a, b);
    } else if constexpr (R == 4) {
        dft4<SIGN>(v[0], v[1], v[2], v[3]);
    } else if constexpr (R == 8) {
        // n = 2 n1 + n2, k = k1 + 4 k2: 4-point DFTs over n1, twiddle W8^(n2 k1), 2-point over n2
        dft4<SIGN>(v[0], v[2], v[4], v[6]);
        dft4<SIGN>(v[1], v[3], v[5], v[7]);
        const float2 o0 = v[1], o1 = mul_w16<2, SIGN>(v[3]), o2 = mul_w16<4, SIGN>(v[5]), o3 = mul_w16<6, SIGN>(v[7]);
        const float2 e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6];
        v[0] = cadd(e0, o0); v[4] = csub(e0, o0);
        v[1] = cadd(e1, o1); v[5] = csub(e1, o1);
        v[2] = cadd(e2, o2); v[6] = csub(e2, o2);
        v[3] = cadd(e3, o3); v[7] = csub(e3, o3);
    } else {
        static_assert(R == 16, "radix");
        // n = 4 n1 + n2, k = k1 + 4 k2
        dft4<SIGN>(v[0], v[4], v[8], v[12]);      // n2 = 0 -> y[0][k1] in v[0], v[4], v[8], v[12]
        dft4<SIGN>(v[1], v[5], v[9], v[13]);      // n2 = 1
        dft4<SIGN>(v[2], v[6], v[10], v[14]);     // n2 = 2
        dft4<SIGN>(v[3], v[7], v[11], v[15]);     // n2 = 3
        // y[n2][k1] sits in v[4 k1 + n2]; multiply by W16^(n2 k1)
        v[5] = mul_w16<1, SIGN>(v[5]);   v[6] = mul_w16<2, SIGN>(v[6]);   v[7] = mul_w16<3, SIGN>(v[7]);
        v[9] = mul_w16<2, SIGN>(v[9]);   v[10] = mul_w16<4, SIGN>(v[10]); v[11] = mul_w16<6, SIGN>(v[11]);
        v[13] = mul_w16<3, SIGN>(v[13]); v[14] = mul_w16<6, SIGN>(v[14]); v[15] = mul_w16<9, SIGN>(v[15]);
        // 4-point DFT over n2 for each k1: inputs v[4 k1 + n2], outputs X[k1 + 4 k2] -> slot 4 k1 + k2
        dft4<SIGN>(v[0], v[1], v[2], v[3]);
        dft4<SIGN>(v[4], v[5], v[6], v[7]);
        dft4<SIGN>(v[8], v[9], v[10], v[11]);
        dft4<SIGN>(v[12], v[13], v[14], v[15]);
        // slot 4 k1 + k2 holds X[k1 + 4 k2]: transpose the 4 x 4 register block
        float2 tmp;
#define RADON_SWAP(i, j) tmp = v[i]; v[i] = v[j]; v[j] = tmp;
        RADON_SWAP(1, 4) RADON_SWAP(2, 8) RADON_SWAP(3, 12) RADON_SWAP(6, 9) RADON_SWAP(7, 13) RADON_SWAP(11, 14)
#undef RADON_SWAP
    }
}

// Barrier between the passes of one FFT.  GROUP == false: the whole CTA (__syncthreads).  GROUP ==
// true: only the TF threads of this FFT (group grp of the CTA, threads grp*TF .. grp*TF + TF - 1):
// a warp-level barrier when the group sits inside one warp, else the named barrier grp + 1, so that
// the FFTs of a CTA drift apart and one group's exchange overlaps another's butterflies.
template <int TF, bool GROUP>
__device__ __forceinline__ void fft_sync(int grp)
{
    if constexpr (!GROUP) __syncthreads();
    else if constexpr (TF <= 32) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "n"(TF) : "memory");
}

// One Stockham pass of radix R; NS = product of the radices already applied.  Register slot
// b + q*NB (NB = 16/R) holds input q of the thread's butterfly b (butterfly index j = b*TF + t).
//   FIRST: inputs are already in v (slot i = element t + i*TF);   otherwise read from s.
//   LAST (R == 16): outputs stay in v (slot u = element t + u*TF); otherwise written to s.
template <int L, int R, int NS, int SIGN, bool FIRST, bool LAST, bool GROUP>
__device__ __forceinline__ void fft_pass(float2 (&v)[16], float2 *s, const float2 *__restrict__ tw, int t, int grp)
{
    constexpr int TF = L / 16, NB = 16 / R, STRIDE = L / R;
    if constexpr (!FIRST) {
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int q = 0; q < R; ++q) v[b + q * NB] = s[FFT_PAD(b * TF + t + q * STRIDE)];
        if constexpr (!LAST) fft_sync<TF, GROUP>(grp);     // everybody has read before anybody overwrites
    }
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        const int j = b * TF + t;
        const int jm = j & (NS - 1);
        float2 x[R];
#pragma unroll
        for (int q = 0; q < R; ++q) x[q] = v[b + q * NB];
        if constexpr (NS > 1) {
            constexpr int TS = L / (NS * R);      // table stride of W_{NS R}
            if constexpr (R == 16) {
                const float2 w1 = __ldg(&tw[jm * TS]), w2 = __ldg(&tw[2 * jm * TS]);
                const float2 w4 = __ldg(&tw[4 * jm * TS]), w8 = __ldg(&tw[8 * jm * TS]);
                const float2 w3 = cmul(w1, w2), w5 = cmul(w1, w4), w6 = cmul(w2, w4), w7 = cmul(w3, w4);
                x[1] = cmul_tw<SIGN>(x[1], w1);   x[2] = cmul_tw<SIGN>(x[2], w2);
                x[3] = cmul_tw<SIGN>(x[3], w3);   x[4] = cmul_tw<SIGN>(x[4], w4);
                x[5] = cmul_tw<SIGN>(x[5], w5);   x[6] = cmul_tw<SIGN>(x[6], w6);
                x[7] = cmul_tw<SIGN>(x[7], w7);   x[8] = cmul_tw<SIGN>(x[8], w8);
                x[9] = cmul_tw<SIGN>(x[9], cmul(w1, w8));    x[10] = cmul_tw<SIGN>(x[10], cmul(w2, w8));
                x[11] = cmul_tw<SIGN>(x[11], cmul(w3, w8));  x[12] = cmul_tw<SIGN>(x[12], cmul(w4, w8));
                x[13] = cmul_tw<SIGN>(x[13], cmul(w5, w8));  x[14] = cmul_tw<SIGN>(x[14], cmul(w6, w8));
                x[15] = cmul_tw<SIGN>(x[15], cmul(w7, w8));
            } else {
#pragma unroll
                for (int q = 1; q < R; ++q) x[q] = cmul_tw<SIGN>(x[q], __ldg(&tw[jm * q * TS]));
            }
        }
        dft_reg<R, SIGN>(x);
        if constexpr (LAST) {
#pragma unroll
            for (int u = 0; u < R; ++u) v[u] = x[u];
        } else {
            const int base = (j - jm) * R + jm;
#pragma unroll
            for (int u = 0; u < R; ++u) s[FFT_PAD(base + u * NS)] = x[u];
        }
    }
    if constexpr (!LAST) fft_sync<TF, GROUP>(grp);
}

// Length-L FFT (SIGN < 0: forward exp(-i..), SIGN > 0: unnormalised inverse).
//   in : v[i] = x[t + i*TF], out: v[i] = X[t + i*TF], TF = L/16, t = 0 .. TF-1.
// s: this FFT's private shared-memory scratch of fft_padded_len(L) float2, free on entry.
// Every thread of the CTA must call it (it contains __syncthreads).  On return other threads
// may still be reading s: the caller synchronises before writing s again.
// GROUP: see fft_sync (then only the TF threads of group grp need to call it together).
template <int L, int SIGN, bool GROUP = false>
__device__ __forceinline__ void fft_reg(float2 (&v)[16], float2 *s, const float2 *__restrict__ tw, int t, int grp = 0)
{
    constexpr int LOG = ilog2_c(L);
    constexpr int R0 = 1 << (LOG % 4);          // first pass: radix 1 (none), 2, 4 or 8
    constexpr int NQ = LOG / 4;                 // then NQ radix-16 passes
    static_assert(NQ >= 1 && NQ <= 3 && L >= 16, "length");
    if constexpr (R0 > 1) {
        fft_pass<L, R0, 1, SIGN, true, false, GROUP>(v, s, tw, t, grp);
        if constexpr (NQ == 1) fft_pass<L, 16, R0, SIGN, false, true, GROUP>(v, s, tw, t, grp);
        if constexpr (NQ == 2) {
            fft_pass<L, 16, R0, SIGN, false, false, GROUP>(v, s, tw, t, grp);
            fft_pass<L, 16, R0 * 16, SIGN, false, true, GROUP>(v, s, tw, t, grp);
        }
        if constexpr (NQ == 3) {
            fft_pass<L, 16, R0, SIGN, false, false, GROUP>(v, s, tw, t, grp);
            fft_pass<L, 16, R0 * 16, SIGN, false, false, GROUP>(v, s, tw, t, grp);
            fft_pass<L, 16, R0 * 256, SIGN, false, true, GROUP>(v, s, tw, t, grp);
        }
    } else {
        if constexpr (NQ == 1) fft_pass<L, 16, 1, SIGN, true, true, GROUP>(v, s, tw, t, grp);
        if constexpr (NQ == 2) {
            fft_pass<L, 16, 1, SIGN, true, false, GROUP>(v, s, tw, t, grp);
            fft_pass<L, 16, 16, SIGN, false, true, GROUP>(v, s, tw, t, grp);
        }
        if constexpr (NQ == 3) {
            fft_pass<L, 16, 1, SIGN, true, false, GROUP>(v, s, tw, t, grp);
            fft_pass<L, 16, 16, SIGN, false, false, GROUP>(v, s, tw, t, grp);
            fft_pass<L, 16, 256, SIGN, false, true, GROUP>(v, s, tw, t, grp);
        }
    }
}

}  // namespace radon
