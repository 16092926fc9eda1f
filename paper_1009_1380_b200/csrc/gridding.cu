// gridding.cu -- the gridding / inverse-gridding kernels of the NUFFT-Radon hot path (sm_100a).
//
//   gather_kernel    F3  inverse gridding, PAPER.md:87 (regular grid -> polar samples)
//   scatter_kernel   A2  gridding, PAPER.md:85 with D == 1 (polar samples -> regular grid)
//                        (+ inside the same launch: the j = 0 samples of all angles summed and
//                        gridded once, DESIGN.md R-tie, and the fixed-order sum of the partial
//                        rectangles of split tiles by the last CTA of a tile to finish)
// (the FFT passes live in fft2d.cu, the projection DFTs in proj.cu)
#include "kernels.h"
#include "async_copy.cuh"
#include "taps.cuh"

#include <atomic>
#include <cstdlib>

namespace radon {

static std::atomic<long long> g_launches{0};
long long launch_count() { return g_launches.load(); }
void count_launch(long long n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
static thread_local bool g_pdl_suppressed = false;
void pdl_suppress(bool on) { g_pdl_suppressed = on; }
bool pdl_enabled()
{
    static const bool on = [] { const char *e = std::getenv("RADON_PDL"); return !(e && e[0] == '0'); }();
    return on && !g_pdl_suppressed;
}

// =====================================================================================
// F3: inverse gridding (gather)
// =====================================================================================
// Persistent CTAs, one per multiprocessor.  A work item = one GT_X x GT_Y tile of the grid
// (+KH halo up/right) and up to GATHER_ROUND_CAP rounds of 32 samples whose footprints start
// inside the tile; the plan assigns items to CTAs (longest first onto the least loaded).
// A producer warp keeps GATHER_STAGES tiles in flight through the copy engine (one bulk copy
// per tile row, rows and columns wrapped mod G; "full" mbarriers count the bytes), so the HBM
// reads never wait for the interpolation; GATHER_WARPS consumer warps take the rounds of the
// CTA's items round-robin (balanced whatever the item sizes) and hand a tile back through an
// "empty" mbarrier.  The 36 taps of a sample are 64-bit shared-memory loads that the
// plan-time schedule made conflict free; slots are fetched two rounds ahead, ray directions one.
constexpr int GATHER_THREADS = (GATHER_WARPS + 1) * 32;
constexpr size_t gather_tile_bytes(int W) { return (size_t)gt_rows(W) * gt_pitch(W) * sizeof(float2); }
constexpr size_t gather_smem(int W) { return GATHER_STAGES * gather_tile_bytes(W); }
static_assert(GT_X % 2 == 0, "bulk copies need 16-byte rows (the pitch GT_X + W is even for the even widths built)");
static_assert(gather_smem(KW_MAX) <= 227 * 1024, "the stages of the widest kernel must fit one CTA");

#ifndef RADON_GATHER_PACKED
#define RADON_GATHER_PACKED 1
#endif
__device__ __forceinline__ uint64_t pack2(float a, float b)
{
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}

__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

template <int KW>
__global__ void __launch_bounds__(GATHER_THREADS, 1)
gather_kernel(const float2 *__restrict__ grid, float2 *__restrict__ polar,
              const GatherCta *__restrict__ items, const int *__restrict__ worker_begin,
              const Slot *__restrict__ slots,
              const double2 *__restrict__ cs, const KbPoly kp,
              int G, int n_det)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t full[GATHER_STAGES], empty[GATHER_STAGES];
    constexpr int GT_PITCH = GT_X + KW, GT_ROWS = GT_Y + KW - 1;          // gt_pitch(KW), gt_rows(KW)
    constexpr size_t GATHER_TILE_BYTES = (size_t)GT_ROWS * GT_PITCH * sizeof(float2);
    pdl_prologue();

    const int it_begin = worker_begin[blockIdx.x], it_end = worker_begin[blockIdx.x + 1];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < GATHER_STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], GATHER_WARPS); }
    }
    __syncthreads();

    if (warp == GATHER_WARPS) {
        // ---- producer: stage the tiles of this CTA's items, GATHER_STAGES ahead ----
        for (int it = it_begin; it < it_end; ++it) {
            const int q = it - it_begin, st = q % GATHER_STAGES;
            const GatherCta item = items[it];
            if (lane == 0) {
                if (q >= GATHER_STAGES) mbar_wait(&empty[st], (uint32_t)((q / GATHER_STAGES - 1) & 1));
                mbar_expect_tx(&full[st], (uint32_t)GATHER_TILE_BYTES);
            }
            __syncwarp();
            float2 *tile = reinterpret_cast<float2 *>(smem_raw + st * GATHER_TILE_BYTES);
            for (int ly = lane; ly < GT_ROWS; ly += 32) {
                const float2 *src = grid + (size_t)((item.ty0 + ly) % G) * G;
                float2 *dst = tile + ly * GT_PITCH;
                int gx = item.tx0, done = 0;                   // tx0 is even, G is even
                while (done < GT_PITCH) {
                    const int n = min(GT_PITCH - done, G - gx);
                    bulk_g2s(dst + done, src + gx, (uint32_t)(n * sizeof(float2)), &full[st]);
                    done += n;
                    gx = 0;
                }
            }
        }
        return;   // every copy is consumed (waited on) by the consumer warps before the CTA ends
    }

    // ---- consumers ----
    const int cd = n_det / 2;
    const double halfG = 0.5 * (double)G;
    // position in the concatenated round sequence of this CTA's items.  Positions only move forward
    // and a slot is loaded right after its position was normalised, so the descriptor of the item a
    // position sits in (round count, first round) is kept in registers and re-read only when the
    // position enters the next item (it was two dependent loads per round).
    struct Pos { int it, r; };
    int c_it = -1, c_rc = 0, c_rb = 0;
    auto norm = [&](Pos p) {
        while (p.it < it_end) {
            if (p.it != c_it) {
                c_it = p.it;
                c_rc = __ldg(&items[p.it].round_count);
                c_rb = __ldg(&items[p.it].round_begin);
            }
            if (p.r < c_rc) break;
            p.r -= c_rc;
            ++p.it;
        }
        return p;
    };
    auto load_slot = [&](const Pos &p) {      // p: the position normalised last
        Slot s;
        s.ak = SLOT_EMPTY; s.lxy = 0;
        if (p.it < it_end) s = slots[((size_t)c_rb + p.r) * 32 + lane];
        return s;
    };
    auto load_dir = [&](const Slot &s) {
        return s.ak != SLOT_EMPTY ? __ldg(&cs[s.ak >> 16]) : make_double2(0.0, 0.0);
    };
    Pos cur = norm(Pos{it_begin, warp});
    Slot sl = load_slot(cur);
    Pos p1 = norm(Pos{cur.it, cur.r + GATHER_WARPS});
    Slot nx = load_slot(p1);
    Pos p2 = norm(Pos{p1.it, p1.r + GATHER_WARPS});
    double2 d = load_dir(sl);
    for (int it = it_begin; it < it_end; ++it) {
        const int q = it - it_begin, st = q % GATHER_STAGES;
        const float2 *tile = reinterpret_cast<const float2 *>(smem_raw + st * GATHER_TILE_BYTES);
        mbar_wait(&full[st], (uint32_t)((q / GATHER_STAGES) & 1));
        while (cur.it == it) {
            const Slot nn = load_slot(p2);
            const double2 dn = load_dir(nx);
            const bool act = sl.ak != SLOT_EMPTY;
            const int a = act ? (int)(sl.ak >> 16) : 0, k = act ? (int)(sl.ak & 0xffff) : 0;
            Taps<KW> tp;
            sample_taps_dir<KW>(d, kp, k, cd, halfG, tp);
            if (act) {
                const float2 *base = tile + (sl.lxy >> 16) * GT_PITCH + (sl.lxy & 0xffff);
#if RADON_GATHER_PACKED
                // packed FMAs (fma.rn.f32x2): re and im of a cell in one instruction, same rounding
                // as two scalar FMAs, half the issue slots of the tap loop
                uint64_t wx2[KW], acc2 = 0ull;
#pragma unroll
                for (int lx = 0; lx < KW; ++lx) wx2[lx] = pack2(tp.wx[lx], tp.wx[lx]);
#pragma unroll
                for (int ly = 0; ly < KW; ++ly) {
                    uint64_t row2 = 0ull;
#pragma unroll
                    for (int lx = 0; lx < KW; ++lx) {
                        const uint64_t v = *reinterpret_cast<const uint64_t *>(&base[ly * GT_PITCH + lx]);
                        asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(row2) : "l"(v), "l"(wx2[lx]));
                    }
                    const uint64_t wy2 = pack2(tp.wy[ly], tp.wy[ly]);
                    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc2) : "l"(row2), "l"(wy2));
                }
                float accr, acci;
                asm("mov.b64 {%0, %1}, %2;" : "=f"(accr), "=f"(acci) : "l"(acc2));
#else
                float accr = 0.f, acci = 0.f;
#pragma unroll
                for (int ly = 0; ly < KW; ++ly) {
                    float rr = 0.f, ri = 0.f;
#pragma unroll
                    for (int lx = 0; lx < KW; ++lx) {
                        const float2 v = base[ly * GT_PITCH + lx];
                        rr = fmaf(v.x, tp.wx[lx], rr);
                        ri = fmaf(v.y, tp.wx[lx], ri);
                    }
                    accr = fmaf(rr, tp.wy[ly], accr);
                    acci = fmaf(ri, tp.wy[ly], acci);
                }
#endif
                // ghost k = n_det (Hermitian-half schedule, even n): F[a, j = -n/2] = conj F[a, j = +n/2]
                if (k == n_det) polar[(size_t)a * n_det] = make_float2(accr, -acci);
                else polar[(size_t)a * n_det + k] = make_float2(accr, acci);
            }
            cur = p1; p1 = p2;
            p2 = norm(Pos{p2.it, p2.r + GATHER_WARPS});
            sl = nx; nx = nn; d = dn;
        }
        if (it + 1 == it_end) pdl_trigger();            // the CTA's last item is done
        // generic-proxy reads of the tile must be ordered before the async-proxy refill
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();                       // every lane has read its taps of this tile
        if (lane == 0) mbar_arrive(&empty[st]);
    }
}

// =====================================================================================
// A2: gridding (scatter) -- CTA-local accumulation in shared memory, no atomics
// =====================================================================================
// A CTA accumulates one SR_X x SR_Y output rectangle in shared memory.  Each warp owns one
// quadrant of it and processes, in rounds of 32 (one sample per lane), every sample whose
// footprint intersects the quadrant, with plain load / FMA / store and the taps clipped to the
// quadrant: warps never share a cell, so there are no atomics and every addition happens in
// a fixed order (bitwise reproducible).  A footprint is processed one ROW at a time (W loads,
// W packed FMAs, W stores, warp barrier); the plan-time schedule guarantees that within a
// row step no two lanes touch the same cell and that every 64-bit access of a half-warp is
// bank-conflict free.  Slots and sample values are prefetched ahead of use.  The finished
// rectangle leaves through the copy engine (bulk shared -> global stores, one per row).
constexpr int SCATTER_THREADS = SCATTER_ITEMS * 32;
// the accumulator of a CTA whose tiles are st_y rows high (a property of the plan: ST_Y or ST_Y_TALL)
constexpr size_t scatter_acc_bytes(int st_y) { return (size_t)(SQ_Y * st_y) * ACC_PITCH * sizeof(float2); }
constexpr size_t SCATTER_SMEM_MAX = scatter_acc_bytes(ST_Y_TALL);
static_assert((ACC_PITCH * sizeof(float2)) % 16 == 0, "bulk stores need 16-byte rows");

__device__ __forceinline__ void bulk_s2g(void *dst, const void *src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 ::"l"(dst), "r"(smem_u32(src)), "r"(bytes) : "memory");
}

// One footprint row of one sample: cell[lx] += (vr, vi) * wx[lx] for the taps whose bit is set in
// `mask` (all loads, then the FMAs, then the stores: the row step of the schedule's disjointness rule).
template <int KW>
__device__ __forceinline__ void scatter_row(uint32_t addr, uint32_t mask, float vr, float vi, const float (&wx)[KW])
{
    uint64_t c[KW];
#pragma unroll
    for (int lx = 0; lx < KW; ++lx) {
        c[lx] = 0ull;
        if (mask & (1u << lx)) asm volatile("ld.shared.b64 %0, [%1];" : "=l"(c[lx]) : "r"(addr + 8u * lx) : "memory");
    }
    const uint64_t v2 = pack2(vr, vi);
#pragma unroll
    for (int lx = 0; lx < KW; ++lx) {
        const uint64_t w2 = pack2(wx[lx], wx[lx]);
        asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(c[lx]) : "l"(v2), "l"(w2));
    }
#pragma unroll
    for (int lx = 0; lx < KW; ++lx)
        if (mask & (1u << lx)) asm volatile("st.shared.b64 [%0], %1;" ::"r"(addr + 8u * lx), "l"(c[lx]) : "memory");
}

// W = 6: one PTX block on a 32-bit shared-window address with immediate offsets: W predicated 64-bit
// loads, 2 W FMAs, W predicated stores, nothing else.
template <>
__device__ __forceinline__ void scatter_row<6>(uint32_t addr, uint32_t mask, float vr, float vi, const float (&wx)[6])
{
    asm volatile(
        "{\n"
        ".reg .pred p0, p1, p2, p3, p4, p5;\n"
        ".reg .b32 t0, t1, t2, t3, t4, t5;\n"
        ".reg .f32 r0, i0, r1, i1, r2, i2, r3, i3, r4, i4, r5, i5;\n"
        "and.b32 t0, %1, 1;\n and.b32 t1, %1, 2;\n and.b32 t2, %1, 4;\n"
        "and.b32 t3, %1, 8;\n and.b32 t4, %1, 16;\n and.b32 t5, %1, 32;\n"
        "setp.ne.b32 p0, t0, 0;\n setp.ne.b32 p1, t1, 0;\n setp.ne.b32 p2, t2, 0;\n"
        "setp.ne.b32 p3, t3, 0;\n setp.ne.b32 p4, t4, 0;\n setp.ne.b32 p5, t5, 0;\n"
        "@p0 ld.shared.v2.f32 {r0, i0}, [%0];\n"
        "@p1 ld.shared.v2.f32 {r1, i1}, [%0+8];\n"
        "@p2 ld.shared.v2.f32 {r2, i2}, [%0+16];\n"
        "@p3 ld.shared.v2.f32 {r3, i3}, [%0+24];\n"
        "@p4 ld.shared.v2.f32 {r4, i4}, [%0+32];\n"
        "@p5 ld.shared.v2.f32 {r5, i5}, [%0+40];\n"
        "fma.rn.f32 r0, %2, %4, r0;\n fma.rn.f32 i0, %3, %4, i0;\n"
        "fma.rn.f32 r1, %2, %5, r1;\n fma.rn.f32 i1, %3, %5, i1;\n"
        "fma.rn.f32 r2, %2, %6, r2;\n fma.rn.f32 i2, %3, %6, i2;\n"
        "fma.rn.f32 r3, %2, %7, r3;\n fma.rn.f32 i3, %3, %7, i3;\n"
        "fma.rn.f32 r4, %2, %8, r4;\n fma.rn.f32 i4, %3, %8, i4;\n"
        "fma.rn.f32 r5, %2, %9, r5;\n fma.rn.f32 i5, %3, %9, i5;\n"
        "@p0 st.shared.v2.f32 [%0], {r0, i0};\n"
        "@p1 st.shared.v2.f32 [%0+8], {r1, i1};\n"
        "@p2 st.shared.v2.f32 [%0+16], {r2, i2};\n"
        "@p3 st.shared.v2.f32 [%0+24], {r3, i3};\n"
        "@p4 st.shared.v2.f32 [%0+32], {r4, i4};\n"
        "@p5 st.shared.v2.f32 [%0+40], {r5, i5};\n"
        "}\n" ::"r"(addr), "r"(mask), "f"(vr), "f"(vi),
        "f"(wx[0]), "f"(wx[1]), "f"(wx[2]), "f"(wx[3]), "f"(wx[4]), "f"(wx[5]) : "memory");
}

// A whole unclipped footprint of one sample (fast rounds: every tap lies inside the quadrant, so
// there are no tap predicates, only `act` for idle lanes).  Row by row: W 64-bit loads, W packed
// FMAs (fma.rn.f32x2: re and im of a cell in one instruction, same rounding as two scalar FMAs),
// W stores, warp barrier.  vrow[ly] = (vr, vi) * wy[ly] packed, w2[lx] = (wx[lx], wx[lx]) packed.
#define RADON_ROW_LD(OFF, R)                                                                          \
    "@p ld.shared.b64 " #R "0, [%0+" #OFF "+0];\n @p ld.shared.b64 " #R "1, [%0+" #OFF "+8];\n"       \
    "@p ld.shared.b64 " #R "2, [%0+" #OFF "+16];\n @p ld.shared.b64 " #R "3, [%0+" #OFF "+24];\n"     \
    "@p ld.shared.b64 " #R "4, [%0+" #OFF "+32];\n @p ld.shared.b64 " #R "5, [%0+" #OFF "+40];\n"
#define RADON_ROW_FMA(V, R)                                                                           \
    "fma.rn.f32x2 " #R "0, " V ", %8, " #R "0;\n fma.rn.f32x2 " #R "1, " V ", %9, " #R "1;\n"          \
    "fma.rn.f32x2 " #R "2, " V ", %10, " #R "2;\n fma.rn.f32x2 " #R "3, " V ", %11, " #R "3;\n"        \
    "fma.rn.f32x2 " #R "4, " V ", %12, " #R "4;\n fma.rn.f32x2 " #R "5, " V ", %13, " #R "5;\n"
#define RADON_ROW_ST(OFF, R)                                                                          \
    "@p st.shared.b64 [%0+" #OFF "+0], " #R "0;\n @p st.shared.b64 [%0+" #OFF "+8], " #R "1;\n"       \
    "@p st.shared.b64 [%0+" #OFF "+16], " #R "2;\n @p st.shared.b64 [%0+" #OFF "+24], " #R "3;\n"     \
    "@p st.shared.b64 [%0+" #OFF "+32], " #R "4;\n @p st.shared.b64 [%0+" #OFF "+40], " #R "5;\n"
#define RADON_WARP_BAR "bar.warp.sync 0xffffffff;\n"
#define RADON_STEP1(O0, V0) RADON_ROW_LD(O0, c) RADON_ROW_FMA(V0, c) RADON_ROW_ST(O0, c) RADON_WARP_BAR
#define RADON_STEP2(O0, V0, O1, V1)                                                                   \
    RADON_ROW_LD(O0, c) RADON_ROW_LD(O1, d) RADON_ROW_FMA(V0, c) RADON_ROW_FMA(V1, d)                 \
    RADON_ROW_ST(O0, c) RADON_ROW_ST(O1, d) RADON_WARP_BAR
#define RADON_STEP3(O0, V0, O1, V1, O2, V2)                                                           \
    RADON_ROW_LD(O0, c) RADON_ROW_LD(O1, d) RADON_ROW_LD(O2, e) RADON_ROW_FMA(V0, c) RADON_ROW_FMA(V1, d) \
    RADON_ROW_FMA(V2, e) RADON_ROW_ST(O0, c) RADON_ROW_ST(O1, d) RADON_ROW_ST(O2, e) RADON_WARP_BAR

// byte offsets of footprint rows 1..5 as literals (they become immediate offsets of the PTX block)
#if RADON_ST_X * RADON_SQ_X == 128
#define RADON_RO1 1040
#define RADON_RO2 2080
#define RADON_RO3 3120
#define RADON_RO4 4160
#define RADON_RO5 5200
#elif RADON_ST_X * RADON_SQ_X == 64
#define RADON_RO1 528
#define RADON_RO2 1056
#define RADON_RO3 1584
#define RADON_RO4 2112
#define RADON_RO5 2640
#else
#error "add the row offsets of this accumulator pitch"
#endif
// widths other than 6: the same row steps from the generic row routine (no tap predicates needed:
// the mask is all ones for an active lane)
template <int KW>
__device__ __forceinline__ void scatter_footprint_fast(uint32_t addr, int act, float vr, float vi, const Taps<KW> &tp)
{
#pragma unroll
    for (int ly = 0; ly < KW; ++ly) {
        scatter_row<KW>(addr + (uint32_t)(ly * ACC_PITCH * (int)sizeof(float2)), act ? ((1u << KW) - 1u) : 0u,
                        vr * tp.wy[ly], vi * tp.wy[ly], tp.wx);
        __syncwarp();
    }
}
template <>
__device__ __forceinline__ void scatter_footprint_fast<6>(uint32_t addr, int act, float vr, float vi, const Taps<6> &tp)
{
    constexpr int KW = 6;
    static_assert(ACC_PITCH * sizeof(float2) == RADON_RO1, "row offsets are written for this pitch");
    uint64_t v[KW], w[KW];
#pragma unroll
    for (int l = 0; l < KW; ++l) {
        v[l] = pack2(vr * tp.wy[l], vi * tp.wy[l]);
        w[l] = pack2(tp.wx[l], tp.wx[l]);
    }
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        ".reg .b64 c0, c1, c2, c3, c4, c5, d0, d1, d2, d3, d4, d5, e0, e1, e2, e3, e4, e5;\n"
        "setp.ne.b32 p, %1, 0;\n"
        "mov.b64 c0, 0;\n mov.b64 c1, 0;\n mov.b64 c2, 0;\n mov.b64 c3, 0;\n mov.b64 c4, 0;\n mov.b64 c5, 0;\n"
        "mov.b64 d0, 0;\n mov.b64 d1, 0;\n mov.b64 d2, 0;\n mov.b64 d3, 0;\n mov.b64 d4, 0;\n mov.b64 d5, 0;\n"
        "mov.b64 e0, 0;\n mov.b64 e1, 0;\n mov.b64 e2, 0;\n mov.b64 e3, 0;\n mov.b64 e4, 0;\n mov.b64 e5, 0;\n"
#if RADON_SC_STEP_ROWS == 1
        RADON_STEP1(0, "%2") RADON_STEP1(RADON_RO1, "%3") RADON_STEP1(RADON_RO2, "%4")
        RADON_STEP1(RADON_RO3, "%5") RADON_STEP1(RADON_RO4, "%6") RADON_STEP1(RADON_RO5, "%7")
#elif RADON_SC_STEP_ROWS == 2
        RADON_STEP2(0, "%2", RADON_RO1, "%3") RADON_STEP2(RADON_RO2, "%4", RADON_RO3, "%5") RADON_STEP2(RADON_RO4, "%6", RADON_RO5, "%7")
#else
        RADON_STEP3(0, "%2", RADON_RO1, "%3", RADON_RO2, "%4") RADON_STEP3(RADON_RO3, "%5", RADON_RO4, "%6", RADON_RO5, "%7")
#endif
        "}\n" ::"r"(addr), "r"(act), "l"(v[0]), "l"(v[1]), "l"(v[2]), "l"(v[3]), "l"(v[4]), "l"(v[5]),
        "l"(w[0]), "l"(w[1]), "l"(w[2]), "l"(w[3]), "l"(w[4]), "l"(w[5]) : "memory");
}

constexpr int DC_CELLS_MAX = (KW_MAX + 1) * (KW_MAX + 1);
// NT threads of one CTA: sum the j = 0 samples of all angles (fixed order) and write the value
// to add to each cell of the (W+1)^2 centre window to dcbuf (cell c: offset ux = c % (W+1) - W/2,
// uy = c / (W+1) - W/2 from DC; zero where nothing is to be added).  part: NT float2 of shared memory.
template <int NT, int KW>
__device__ __forceinline__ void dc_compute(const float2 *__restrict__ polar, const KbPoly &kp, int n_det, int n_angles, int half,
                                           float2 *part, float2 *__restrict__ dcbuf)
{
    const int t = threadIdx.x, cd = n_det / 2;
    float sr = 0.f, si = 0.f;
    for (int a0 = 0; a0 < n_angles; a0 += 8 * NT) {              // 8 independent loads in flight
        float2 v[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int a = a0 + q * NT + t;
            v[q] = a < n_angles ? __ldg(&polar[(size_t)a * n_det + cd]) : make_float2(0.f, 0.f);
        }
#pragma unroll
        for (int q = 0; q < 8; ++q) { sr += v[q].x; si += v[q].y; }
    }
    part[t] = make_float2(sr, si);
    __syncthreads();
    for (int h = NT / 2; h > 0; h >>= 1) {
        if (t < h) { part[t].x += part[t + h].x; part[t].y += part[t + h].y; }
        __syncthreads();
    }
    const float2 V = part[0];
    constexpr int DC_CELLS = (KW + 1) * (KW + 1);
    float wa[KW], wb[KW];
    kb_poly_weights<KW>(kp, 0.f, wa);
    kb_poly_weights<KW>(kp, 1.f, wb);
    auto tap = [](const float (&w)[KW], int l) {
        float r = 0.f;
#pragma unroll
        for (int q = 0; q < KW; ++q) r = (q == l) ? w[q] : r;
        return r;
    };
    for (int c = t; c < DC_CELLS; c += NT) {
        const int ux = c % (KW + 1) - KW / 2, uy = c / (KW + 1) - KW / 2;     // cell offset from DC: -W/2 .. W/2
        const float a2 = tap(wa, ux + KW / 2) * tap(wa, uy + KW / 2);           // taps -W/2 .. W/2-1
        const float b2 = tap(wb, ux + KW / 2 - 1) * tap(wb, uy + KW / 2 - 1);   // taps -W/2+1 .. W/2
        float2 add = make_float2(0.f, 0.f);
        if (half) {
            if (uy >= 0) add = make_float2(0.5f * V.x * (a2 + b2), 0.5f * V.y * (a2 - b2));
        } else {
            add = make_float2(V.x * a2, V.y * a2);
        }
        dcbuf[c] = add;
    }
}

// Fixed-order sum of the partial rectangles of a merge job (split rectangle and / or centre
// window), rows [y_begin, y_end) of the rectangle: NT threads, two cells (16 bytes) per access,
// four pairs times four slots in flight per thread.  The order of the additions is the slot
// order, whoever runs this: bitwise reproducible.  dcbuf: the summed j = 0 samples on the
// (W+1)^2 centre window (DESIGN.md R-tie).
template <int NT>
__device__ __forceinline__ void merge_rows(const MergeJob &j, int y_begin, int y_end, const float2 *__restrict__ scratch,
                                           float2 *__restrict__ grid, int G, const float2 *__restrict__ dcbuf, int KW, int slot_cells)
{
    const int ppr = j.rw >> 1, p_begin = ppr * y_begin, p_end = ppr * y_end;        // rw is even (check_schedules)
    const float4 *src = reinterpret_cast<const float4 *>(scratch + (size_t)j.first_slot * slot_cells);
    const int SLOT4 = slot_cells / 2;
    constexpr int ROW4 = SR_X / 2;
    const bool has_dc = j.expected > j.n_slots;
    for (int i0 = p_begin + threadIdx.x; i0 < p_end; i0 += 4 * NT) {
        float4 sum[4];
        int off[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int i = min(i0 + q * NT, p_end - 1), y = i / ppr, x = i - y * ppr;
            off[q] = y * ROW4 + x;
            sum[q] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        for (int s0 = 0; s0 < j.n_slots; s0 += 4) {
            float4 v[4][4];
#pragma unroll
            for (int t = 0; t < 4; ++t)
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    v[t][q] = (s0 + t < j.n_slots) ? __ldcg(&src[(size_t)(s0 + t) * SLOT4 + off[q]])
                                                   : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
            for (int t = 0; t < 4; ++t)
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    sum[q].x += v[t][q].x; sum[q].y += v[t][q].y; sum[q].z += v[t][q].z; sum[q].w += v[t][q].w;
                }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int i = i0 + q * NT;
            if (i >= p_end) continue;
            const int y = i / ppr, x = 2 * (i - y * ppr);
            if (has_dc) {
                const int uy = j.ry0 + y - G / 2, ux = j.rx0 + x - G / 2;
                if (uy >= -KW / 2 && uy <= KW / 2) {
                    if (ux >= -KW / 2 && ux <= KW / 2) {
                        const float2 d = __ldcg(&dcbuf[(uy + KW / 2) * (KW + 1) + ux + KW / 2]);
                        sum[q].x += d.x; sum[q].y += d.y;
                    }
                    if (ux + 1 >= -KW / 2 && ux + 1 <= KW / 2) {
                        const float2 d = __ldcg(&dcbuf[(uy + KW / 2) * (KW + 1) + ux + 1 + KW / 2]);
                        sum[q].z += d.x; sum[q].w += d.y;
                    }
                }
            }
            *reinterpret_cast<float4 *>(grid + (size_t)(j.ry0 + y) * G + j.rx0 + x) = sum[q];
        }
    }
}

// A CTA's part in merge job `job` (all NT threads call it, after this CTA's contribution to the
// job is complete and fenced).  Three counters per job: arrivals, row chunks claimed, departures.
// The job is READY once all `expected` contributions have arrived; from then on any of its CTAs
// claims row chunks and merges them.  The CTA that makes the job ready always drains the chunk
// counter, so the merge completes whoever helps; the others (the CTAs of a split rectangle get
// the same number of rounds and finish together) wait a BOUNDED time for the job to become
// ready, so that the rows are merged side by side instead of by the last CTA alone, and leave
// without helping when the bound expires.  The last CTA to depart re-arms the counters for the
// next launch (also under graph replay: no host-side epoch).
constexpr int MERGE_COUNTERS = MERGE_COUNTERS_PER_JOB;   // ints per job: arrivals, chunks, departures, pad
#ifndef RADON_MERGE_WAIT_NS
#define RADON_MERGE_WAIT_NS 20000
#endif
template <int NT>
__device__ __forceinline__ void join_merge(int job, bool wait, const MergeJob *__restrict__ jobs, int *__restrict__ tickets,
                                           const float2 *__restrict__ scratch, float2 *__restrict__ grid, int G,
                                           const float2 *__restrict__ dcbuf, int *s_flag, int KW, int slot_cells)
{
    int *cnt = tickets + job * MERGE_COUNTERS;
    const MergeJob j = jobs[job];
    __syncthreads();                              // every thread's writes are fenced
    if (threadIdx.x == 0) {
        bool ready = atomicAdd(&cnt[0], 1) == j.expected - 1;
        if (!ready && wait) {
            unsigned long long t0, t1;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
            do {
                __nanosleep(256);
                int a;
                asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(a) : "l"(&cnt[0]) : "memory");
                ready = a >= j.expected;
                asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
            } while (!ready && t1 - t0 < (unsigned long long)RADON_MERGE_WAIT_NS);
        }
        *s_flag = ready ? 1 : 0;
    }
    __syncthreads();
    if (*s_flag) {
        __threadfence();                          // the other CTAs' slots, fenced before their arrivals
        // chunks of rows: about two per contributing CTA, an even number of rows each
        int rows = max(2, (j.rh / (2 * j.n_slots)) & ~1);
        const int n_chunks = (j.rh + rows - 1) / rows;
        for (;;) {
            __syncthreads();
            if (threadIdx.x == 0) *s_flag = atomicAdd(&cnt[1], 1);
            __syncthreads();
            const int c = *s_flag;
            if (c >= n_chunks) break;
            merge_rows<NT>(j, c * rows, min(j.rh, (c + 1) * rows), scratch, grid, G, dcbuf, KW, slot_cells);
        }
    }
    __syncthreads();
    if (threadIdx.x == 0 && atomicAdd(&cnt[2], 1) == j.expected - 1) {
        cnt[0] = 0; cnt[1] = 0; cnt[2] = 0;       // everybody has left: nobody reads the counters any more
    }
}

struct DcJobs { int n; int job[MAX_DC_JOBS]; };

template <int KW>
__global__ void __launch_bounds__(SCATTER_THREADS, SCATTER_CTAS_PER_SM)
scatter_kernel(const float2 *__restrict__ polar, float2 *__restrict__ grid, float2 *__restrict__ scratch,
               const ScatterCta *__restrict__ ctas, const Slot *__restrict__ slots,
               const double2 *__restrict__ cs, const KbPoly kp,
               int G, int n_det, int nyq_split, float2 *__restrict__ dcbuf, int n_angles, int half,
               const MergeJob *__restrict__ jobs, int *__restrict__ tickets, const DcJobs dcj, int st_y)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float2 *acc = reinterpret_cast<float2 *>(smem_raw);
    __shared__ int s_flag;
    const int slot_cells = SR_X * SQ_Y * st_y;      // cells of a partial rectangle in scratch
    pdl_prologue();
    if (blockIdx.x == 0) {
        // CTA 0: the j = 0 samples of all angles, summed (fixed order) while the others grid; the
        // footprint of the sum is added by the merge of the centre rectangles (DESIGN.md R-tie)
        dc_compute<SCATTER_THREADS, KW>(polar, kp, n_det, n_angles, half, acc, dcbuf);
        __threadfence();
        for (int q = 0; q < dcj.n; ++q)
            join_merge<SCATTER_THREADS>(dcj.job[q], false, jobs, tickets, scratch, grid, G, dcbuf, &s_flag, KW, slot_cells);
        return;
    }
    __shared__ ScatterCta cta;

    if (threadIdx.x < sizeof(ScatterCta) / 4)
        reinterpret_cast<int *>(&cta)[threadIdx.x] = reinterpret_cast<const int *>(&ctas[blockIdx.x - 1])[threadIdx.x];
    __syncthreads();

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int cd = n_det / 2;
    const double halfG = 0.5 * (double)G;
    const ScatterItem item = cta.items[warp];
    const Slot *my = slots + (size_t)item.round_begin * 32 + lane;
    const int nr = item.round_count;
    // software pipeline (the slot stream comes from HBM, the sample values from L2): slots are
    // fetched four rounds ahead, sample values and ray directions two rounds ahead
    auto load_slot = [&](int r) {
        Slot s;
        s.ak = SLOT_EMPTY; s.lxy = 0;
        if (r < nr) s = my[(size_t)r * 32];
        return s;
    };
    auto load_value = [&](const Slot &s, float2 &v, double2 &d) {
        v = make_float2(0.f, 0.f);
        d = make_double2(0.0, 0.0);
        if (s.ak != SLOT_EMPTY) {
            const int k = (int)(s.ak & 0xffff);
            v = __ldg(&polar[(size_t)(s.ak >> 16) * n_det + (k == n_det ? 0 : k)]);
            d = __ldg(&cs[s.ak >> 16]);
        }
    };
    Slot s0 = load_slot(0), s1 = load_slot(1), s2 = load_slot(2), s3 = load_slot(3);
    {   // zero the accumulator while those loads are in flight
        float4 *z = reinterpret_cast<float4 *>(acc);
        for (int i = threadIdx.x; i < SQ_Y * st_y * ACC_PITCH / 2; i += SCATTER_THREADS)
            z[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    float2 v0, v1;
    double2 d0, d1;
    load_value(s0, v0, d0);
    load_value(s1, v1, d1);
    __syncthreads();

    // shared-window address of slot (0,0); never dereferenced outside the quadrant
    constexpr int KH = KW - 1;
    const uint32_t origin = smem_u32(acc) + (uint32_t)(((item.sy0 - KH) * ACC_PITCH + (item.sx0 - KH)) * (int)sizeof(float2));
    for (int r = 0; r < nr; ++r) {
        const Slot s4 = load_slot(r + 4);
        float2 v2;
        double2 d2;
        load_value(s2, v2, d2);
        const bool act = s0.ak != SLOT_EMPTY;
        const int k0 = (int)(s0.ak & 0xffff);
        // Hermitian-half schedule, even n: the unpaired Nyquist sample k = 0 (j = -n/2) and its
        // ghost k = n (j = +n/2) carry half the value each, the ghost conjugated.  Applied here,
        // at the point of use, so that the prefetched load stays off the critical path.
        if (nyq_split && (k0 == 0 || k0 == n_det)) v0 = make_float2(0.5f * v0.x, k0 == 0 ? 0.5f * v0.y : -0.5f * v0.y);
        Taps<KW> tp;
        sample_taps_dir<KW>(d0, kp, k0, cd, halfG, tp);
        const int bx = (int)(s0.lxy & 0xffff), by = (int)(s0.lxy >> 16);   // biased by KH
        const uint32_t base = origin + (uint32_t)((by * ACC_PITCH + bx) * (int)sizeof(float2));
        if (RADON_SC_FAST && r < item.fast_count) {   // warp-uniform: footprints wholly inside the quadrant
            scatter_footprint_fast<KW>(base, act ? 1 : 0, v0.x, v0.y, tp);
        } else {
        // taps inside the quadrant: KH <= bx + lx < KH + sw, likewise rows -> bit masks
        const int xlo = min(max(KH - bx, 0), KW), xhi = min(max(KH + item.sw - bx, 0), KW);
        const int ylo = min(max(KH - by, 0), KW), yhi = min(max(KH + item.sh - by, 0), KW);
        const uint32_t xmask = act ? (((1u << xhi) - 1u) & ~((1u << xlo) - 1u)) : 0u;
        const uint32_t ymask = ((1u << yhi) - 1u) & ~((1u << ylo) - 1u);
#pragma unroll
        for (int ly = 0; ly < KW; ++ly) {
            const uint32_t m = (ymask & (1u << ly)) ? xmask : 0u;
            scatter_row<KW>(base + (uint32_t)(ly * ACC_PITCH * (int)sizeof(float2)), m,
                        v0.x * tp.wy[ly], v0.y * tp.wy[ly], tp.wx);
            __syncwarp();   // row steps of different lanes may touch the same cells
        }
        }
        s0 = s1; s1 = s2; s2 = s3; s3 = s4;
        v0 = v1; v1 = v2; d0 = d1; d1 = d2;
    }

    pdl_trigger();
    // flush: the rectangle is written exactly once, by the copy engine
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> async proxy
    __syncthreads();
    float2 *dst;
    int dpitch;
    if (cta.partial_slot >= 0) { dst = scratch + (size_t)cta.partial_slot * slot_cells; dpitch = SR_X; }
    else { dst = grid + (size_t)cta.ry0 * G + cta.rx0; dpitch = G; }
    for (int y = threadIdx.x; y < cta.rh; y += SCATTER_THREADS)          // one bulk store per row
        bulk_s2g(dst + (size_t)y * dpitch, acc + y * ACC_PITCH, (uint32_t)(cta.rw * sizeof(float2)));
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    if (cta.job < 0) {
        asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // shared memory must outlive the reads
        return;
    }
    // partial rectangle: its writes must have landed, and be visible device-wide, before the ticket
    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    asm volatile("fence.proxy.async;" ::: "memory");
    __threadfence();
    join_merge<SCATTER_THREADS>(cta.job, true, jobs, tickets, scratch, grid, G, dcbuf, &s_flag, KW, slot_cells);
}

// The j = 0 samples (k = n/2) of all angles sit at kappa = (0,0) and share one footprint, so
// they are left out of the scatter schedules: CTA 0 sums their values (fixed order) and the
// footprint of the sum is added once, by the merge of the centre rectangles (no atomics).
// Full grid: V * wA(kx) wA(ky), wA = the rule-A taps [-W/2, W/2) of an exact tie (delta = 0).
// Hermitian half (rows ky >= 0 only; the rows below are implied by symmetry): the Hermitian
// part of that footprint, (V wA(kx) wA(ky) + conj(V) wB(kx) wB(ky)) / 2, wB(u) = wA(-u) the
// mirrored taps (-W/2, W/2] (delta = 1) -- what the full gridding followed by Re{.} computes
// (reading R-tie).
int launch_gather(const DevicePlan &p, bool half, const float2 *grid, float2 *polar, cudaStream_t st)
{
    const DevicePlan::Sched &q = p.sched[half ? 1 : 0];
    if (q.n_gather_ctas == 0) return 0;
    RADON_FOR_W(p.W, launch_pdl(p.pdl, gather_kernel<WW>, q.n_gather_workers, GATHER_THREADS, gather_smem(WW), st,
        grid, polar, q.gather_ctas, q.gather_worker_begin, q.gather_slots, p.cs, p.kb, p.G, p.n_det);)
    count_launch();
    return 0;
}

int launch_scatter(const DevicePlan &p, bool half, const float2 *polar, float2 *grid, float2 *scratch,
                   float2 *dcbuf, int *tickets, cudaStream_t st)
{
    const DevicePlan::Sched &q = p.sched[half ? 1 : 0];
    const int nyq = (half && (p.n_det & 1) == 0) ? 1 : 0;
    DcJobs dcj;
    dcj.n = q.n_dc_jobs;
    for (int i = 0; i < MAX_DC_JOBS; ++i) dcj.job[i] = q.dc_jobs[i];
    // CTA 0 sums the j = 0 samples; CTA b > 0 grids scatter_ctas[b - 1] (heaviest first)
    RADON_FOR_W(p.W, launch_pdl(p.pdl, scatter_kernel<WW>, q.n_scatter_ctas + 1, SCATTER_THREADS, scatter_acc_bytes(p.st_y), st,
        polar, grid, scratch, q.scatter_ctas, q.scatter_slots, p.cs, p.kb, p.G, p.n_det, nyq,
        dcbuf, p.n_angles, half ? 1 : 0, q.merge_jobs, tickets, dcj, p.st_y);)
    count_launch();
    return 0;
}

int init_kernel_attributes()
{
    if (set_smem(gather_kernel<4>, gather_smem(4)) || set_smem(gather_kernel<6>, gather_smem(6)) ||
        set_smem(gather_kernel<8>, gather_smem(8))) return -1;
    if (set_smem(scatter_kernel<4>, SCATTER_SMEM_MAX) || set_smem(scatter_kernel<6>, SCATTER_SMEM_MAX) ||
        set_smem(scatter_kernel<8>, SCATTER_SMEM_MAX)) return -1;
    return 0;
}

}  // namespace radon
