// plan_device.cu -- P3 on the device: sample binning into grid tiles and the packing of every
// tile's samples into conflict-free rounds (the plan-time work that takes the place of the
// paper's load-balanced bins), as CUDA kernels.
//
//   count_regions_kernel   one warp per tile: which polar samples (and which of their periodic
//                          images) have a footprint in the tile -- found from the Fourier-slice
//                          geometry itself: along one radial line the base cell
//                          ceil(j d + G/2 - W/2) is monotone in j, so a tile sees an interval of
//                          j per angle; no global sort, no atomics, and the enumeration order
//                          (image, angle, j) is the same on every run.
//   fill_pack_kernel       one warp per LIST (a gather tile, or one of the K shares of a scatter
//                          tile): enumerates the tile again, keeps its share (inside footprints
//                          first, clipped ones after), and packs it into rounds of 32 lanes with
//                          the rule of plan_host.cpp's build_rounds: first fit in list order,
//                          distinct bank pairs per half-warp, (scatter) no two lanes of a round
//                          with the same base row and base columns closer than W, then idle
//                          lanes take candidates whose bank pair is used once.
//   compact_rounds_kernel  copies the rounds of every list to their final place.
// The host keeps what is small: tile tables, the split factor K of heavy tiles, prefix sums,
// the assignment of gather items to persistent CTAs.  check_schedules (plan_host.cpp) verifies a
// device-built schedule exactly as it verifies a host-built one.
#include "kernels.h"
#include "plan_device.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>

namespace radon {

struct SampleSet {              // which (a, k) a schedule covers
    int n_angles, n_det, G;
    int k0, k1;                 // k in [k0, k1); k == n_det is the Nyquist ghost (j = +n/2)
    int skip_k;                 // left out (scatter: j = 0), or -1
    int W;                      // kernel width
};

__device__ __forceinline__ void base_cell(const double2 d, int j, double halfG, int KW, int &x0, int &y0)
{
    // the same fp64 expressions as Geometry::base and sample_taps_dir: bit-identical tap selection
    x0 = (int)ceil(fma((double)j, d.x, halfG) - 0.5 * KW);
    y0 = (int)ceil(fma((double)j, d.y, halfG) - 0.5 * KW);
}

// j interval (conservative, two cells of slack) in which ceil(j d + c) can lie in [lo, hi]
__device__ __forceinline__ void j_interval(double d, double c, int lo, int hi, int &jlo, int &jhi)
{
    const double A = (double)lo - 2.0 - c, B = (double)hi + 1.0 - c;      // j d in [A, B]
    if (fabs(d) < 1e-9) {
        if (A > 0.0 || B < 0.0) { jlo = 1; jhi = 0; }
        return;                                                           // every j
    }
    const double u = A / d, v = B / d;
    jlo = max(jlo, (int)fmax(floor(fmin(u, v)) - 1.0, -1e9));
    jhi = min(jhi, (int)fmin(ceil(fmax(u, v)) + 1.0, 1e9));
}

// Calls f(ak, lx, ly, image) for every candidate of `r` on angle a, in j order, for image (sx, sy).
template <typename F>
__device__ __forceinline__ void for_candidates(const PackRegion &r, const SampleSet &s, const double2 d, int a,
                                               int sx, int sy, F f)
{
    const int cd = s.n_det / 2, KW = s.W;
    const double halfG = 0.5 * (double)s.G;
    int jlo = s.k0 - cd, jhi = s.k1 - 1 - cd;
    j_interval(d.x, halfG - 0.5 * KW + (double)sx * s.G, r.rx0 - r.lo, r.rx0 + r.rw - 1, jlo, jhi);
    j_interval(d.y, halfG - 0.5 * KW + (double)sy * s.G - (double)r.oy, r.ry0 - r.lo, r.ry0 + r.rh - 1, jlo, jhi);
    for (int j = jlo; j <= jhi; ++j) {
        const int k = j + cd;
        if (k == s.skip_k) continue;
        int x0, y0;
        base_cell(d, j, halfG, KW, x0, y0);
        const int bx = x0 + sx * s.G, by = y0 + sy * s.G - r.oy;
        if (bx < r.rx0 - r.lo || bx >= r.rx0 + r.rw || by < r.ry0 - r.lo || by >= r.ry0 + r.rh) continue;
        if (r.lo == 0 && (bx < 0 || bx >= s.G || by < 0 || by >= s.G)) continue;     // gather: one image per sample
        f(((uint32_t)a << 16) | (uint32_t)k, bx - (r.rx0 - r.lo), by - (r.ry0 - r.lo));
    }
}

__device__ __forceinline__ bool cand_inside(const PackRegion &r, int lx, int ly)
{
    return r.lo == 0 || (lx >= r.lo && lx <= r.rw - 1 && ly >= r.lo && ly <= r.rh - 1);     // scatter: lo = W - 1
}

// ---- pass 1: count the candidates of every region ---------------------------------------------
constexpr int PLAN_WARPS = 4;
__global__ void __launch_bounds__(PLAN_WARPS * 32)
count_regions_kernel(PackRegion *__restrict__ regions, int n_regions, const double2 *__restrict__ cs, const SampleSet s)
{
    __shared__ int rowcnt[PLAN_WARPS][SB_H_MAX > GT_ROWS_MAX ? SB_H_MAX : GT_ROWS_MAX];
    const int ri = blockIdx.x * PLAN_WARPS + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (ri >= n_regions) return;
    const PackRegion r = regions[ri];
    int *rc = rowcnt[threadIdx.x >> 5];
    constexpr int NROW = SB_H_MAX > GT_ROWS_MAX ? SB_H_MAX : GT_ROWS_MAX;
    for (int i = lane; i < NROW; i += 32) rc[i] = 0;
    __syncwarp();
    int n_in = 0, n_cl = 0;
    for (int sy = -1; sy <= 1; ++sy)
        for (int sx = -1; sx <= 1; ++sx)
            for (int a = lane; a < s.n_angles; a += 32)
                for_candidates(r, s, __ldg(&cs[a]), a, sx, sy, [&](uint32_t, int lx, int ly) {
                    if (cand_inside(r, lx, ly)) ++n_in; else ++n_cl;
                    if (r.lo) atomicAdd(&rc[ly], 1);
                });
    __syncwarp();
    int mrow = 0;
    for (int i = lane; i < NROW; i += 32) mrow = max(mrow, rc[i]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        n_in += __shfl_xor_sync(0xffffffffu, n_in, o);
        n_cl += __shfl_xor_sync(0xffffffffu, n_cl, o);
        mrow = max(mrow, __shfl_xor_sync(0xffffffffu, mrow, o));
    }
    if (lane == 0) { regions[ri].n_in = n_in; regions[ri].n_cl = n_cl; regions[ri].max_row = mrow; }
}

// ---- pass 2: one warp per list -------------------------------------------------------------------
struct RoundState {
    uint32_t mask[2], twice[2];
    int cnt[2];
};

// occupancy of the round: one 128-bit row per base row (bit = base column no other lane may take)
struct OccRows { unsigned long long w[(SB_H_MAX > GT_ROWS_MAX ? SB_H_MAX : GT_ROWS_MAX)][2]; };

__device__ __forceinline__ bool occ_overlaps(const OccRows &o, int lx, int ly)
{
    return (o.w[ly][lx >> 6] >> (lx & 63)) & 1ull;
}
__device__ __forceinline__ void occ_mark(OccRows &o, int lx, int ly, int KH)       // one lane
{
    const int lo = max(lx - KH, 0), hi = min(lx + KH, 127);
    for (int x = lo; x <= hi; ++x) o.w[ly][x >> 6] |= 1ull << (x & 63);
}

__global__ void __launch_bounds__(32)
fill_pack_kernel(PackList *__restrict__ lists, const PackRegion *__restrict__ regions, const double2 *__restrict__ cs,
                 const SampleSet s, Slot *__restrict__ cand_all, Slot *__restrict__ tmp_slots, int pitch, int disjoint)
{
    __shared__ OccRows occ;
    const int lane = threadIdx.x;
    PackList L = lists[blockIdx.x];
    const PackRegion r = regions[L.region];
    Slot *cand = cand_all + L.cand_begin;
    const int K = L.K, kk = L.kk;
    const int n_in_sub = (r.n_in > kk) ? (r.n_in - kk + K - 1) / K : 0;
    const int n_cl_sub = (r.n_cl > kk) ? (r.n_cl - kk + K - 1) / K : 0;
    const int n = n_in_sub + n_cl_sub;

    // -- enumerate the tile, keep this list's share: position q of the tile's inside (clipped)
    //    candidates goes to list q % K, place q / K (after the inside ones for the clipped)
    int q_in = 0, q_cl = 0;                                  // warp-uniform running counts
    for (int sy = -1; sy <= 1; ++sy)
        for (int sx = -1; sx <= 1; ++sx)
            for (int a0 = 0; a0 < s.n_angles; a0 += 32) {
                const int a = a0 + lane;
                int c_in = 0, c_cl = 0;
                double2 d = make_double2(0.0, 0.0);
                if (a < s.n_angles) {
                    d = __ldg(&cs[a]);
                    for_candidates(r, s, d, a, sx, sy, [&](uint32_t, int lx, int ly) {
                        if (cand_inside(r, lx, ly)) ++c_in; else ++c_cl;
                    });
                }
                int p_in = c_in, p_cl = c_cl;                // inclusive scans over the lanes
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int u = __shfl_up_sync(0xffffffffu, p_in, o), v = __shfl_up_sync(0xffffffffu, p_cl, o);
                    if (lane >= o) { p_in += u; p_cl += v; }
                }
                const int t_in = __shfl_sync(0xffffffffu, p_in, 31), t_cl = __shfl_sync(0xffffffffu, p_cl, 31);
                if (a < s.n_angles && (c_in | c_cl)) {
                    int my_in = q_in + p_in - c_in, my_cl = q_cl + p_cl - c_cl;
                    for_candidates(r, s, d, a, sx, sy, [&](uint32_t ak, int lx, int ly) {
                        Slot e;
                        e.ak = ak; e.lxy = (uint32_t)lx | ((uint32_t)ly << 16);
                        if (cand_inside(r, lx, ly)) {
                            if (my_in % K == kk) cand[my_in / K] = e;
                            ++my_in;
                        } else {
                            if (my_cl % K == kk) cand[n_in_sub + my_cl / K] = e;
                            ++my_cl;
                        }
                    });
                }
                q_in += t_in; q_cl += t_cl;
            }
    __syncwarp();

    // -- pack: first fit in list order (plan_host.cpp build_rounds).  The remaining candidates
    //    live in cand[begin, n); after a round the scanned prefix is compacted towards its end.
    Slot *out = tmp_slots + (size_t)L.tmp_round_begin * 32;
    int begin = 0, rounds = 0, n_fast = 0, filled = 0;
    bool fast_open = true, overflow = false;
    while (begin < n) {
        if (rounds >= L.round_cap) { overflow = true; break; }
        if (disjoint) {
            unsigned long long *z = &occ.w[0][0];
            for (int i = lane; i < (int)(sizeof(OccRows) / 8); i += 32) z[i] = 0ull;
        }
        Slot *row = out + (size_t)rounds * 32;
        row[lane].ak = SLOT_EMPTY; row[lane].lxy = 0;
        __syncwarp();
        RoundState st;
        st.mask[0] = st.mask[1] = st.twice[0] = st.twice[1] = 0u; st.cnt[0] = st.cnt[1] = 0;
        bool all_in = true;
        int scanned_end = begin;
        for (int pass = 0; pass < 2; ++pass) {
            if (st.cnt[0] + st.cnt[1] == 32) break;
            for (int i0 = begin; i0 < n; i0 += 32) {
                const int i = i0 + lane;
                Slot c;
                c.ak = SLOT_EMPTY; c.lxy = 0;
                if (i < n) c = cand[i];
                const int lx = (int)(c.lxy & 0xffff), ly = (int)(c.lxy >> 16);
                const uint32_t res = 1u << ((ly * pitch + lx) & 15);
                bool pending = c.ak != SLOT_EMPTY;           // accepted entries were marked empty
                for (;;) {
                    int h = -1;
                    if (pending && !(disjoint && occ_overlaps(occ, lx, ly))) {
                        if (pass == 0) {
                            if (st.cnt[0] < 16 && !(st.mask[0] & res)) h = 0;
                            else if (st.cnt[1] < 16 && !(st.mask[1] & res)) h = 1;
                        } else {
                            if (st.cnt[0] < 16 && !(st.twice[0] & res)) h = 0;
                            else if (st.cnt[1] < 16 && !(st.twice[1] & res)) h = 1;
                        }
                    }
                    const unsigned ok = __ballot_sync(0xffffffffu, h >= 0);
                    if (!ok) break;
                    const int win = __ffs(ok) - 1;           // the first feasible candidate in list order
                    const int wh = __shfl_sync(0xffffffffu, h, win);
                    const uint32_t wres = __shfl_sync(0xffffffffu, res, win);
                    if (lane == win) {
                        row[wh * 16 + st.cnt[wh]] = c;
                        cand[i].ak = SLOT_EMPTY;
                        if (disjoint) occ_mark(occ, lx, ly, s.W - 1);
                        pending = false;
                    }
                    all_in = all_in && __shfl_sync(0xffffffffu, (int)cand_inside(r, lx, ly), win);
                    if (pass == 0 || !(st.mask[wh] & wres)) st.mask[wh] |= wres; else st.twice[wh] |= wres;
                    st.cnt[wh]++;
                    __syncwarp();
                    if (lane < win) pending = false;         // rejected for this round: the state only tightens
                    if (st.cnt[0] + st.cnt[1] == 32) break;
                }
                scanned_end = max(scanned_end, min(n, i0 + 32));
                if (st.cnt[0] + st.cnt[1] == 32) break;
            }
        }
        filled += st.cnt[0] + st.cnt[1];
        if (fast_open && all_in) ++n_fast; else fast_open = false;
        ++rounds;
        // compact the scanned prefix [begin, scanned_end) towards its end, order kept
        int wr = scanned_end;
        for (int hi = scanned_end; hi > begin; hi -= 32) {
            const int i = hi - 32 + lane;                    // chunk [hi - 32, hi), may start below begin
            Slot c;
            c.ak = SLOT_EMPTY; c.lxy = 0;
            if (i >= begin) c = cand[i];
            const unsigned alive = __ballot_sync(0xffffffffu, c.ak != SLOT_EMPTY);
            const int after = __popc(alive >> lane) - 1;    // alive lanes above this one
            __syncwarp();
            if (c.ak != SLOT_EMPTY) cand[wr - 1 - after] = c;
            wr -= __popc(alive);
            __syncwarp();
        }
        begin = wr;
    }
    if (lane == 0) {
        lists[blockIdx.x].n = n;
        lists[blockIdx.x].n_rounds = rounds;
        lists[blockIdx.x].n_fast = n_fast;
        lists[blockIdx.x].filled = filled;
        lists[blockIdx.x].overflow = overflow ? 1 : 0;
    }
}

// ---- pass 3: rounds of every list -> their final place ------------------------------------------
__global__ void __launch_bounds__(256)
compact_rounds_kernel(const PackList *__restrict__ lists, int n_lists, Slot *__restrict__ slots)
{
    const int li = blockIdx.x;
    if (li >= n_lists) return;
    const PackList L = lists[li];
    Slot *dst = slots + (size_t)L.round_begin * 32;
    for (int i = threadIdx.x; i < L.n_rounds * 32; i += blockDim.x) dst[i] = L.src[i];
}

// ---- host driver ----------------------------------------------------------------------------------
#define PD_TRY(expr)                                   \
    do {                                               \
        if ((expr) != cudaSuccess) { rc = -1; goto done; } \
    } while (0)

int device_pack(const double2 *d_cs, const DevicePackParams &prm, std::vector<PackRegion> &regions,
                std::vector<PackList> &lists, Slot **d_slots_out, long long *n_rounds_out)
{
    int rc = 0;
    SampleSet s;
    s.n_angles = prm.n_angles; s.n_det = prm.n_det; s.G = prm.G; s.k0 = prm.k0; s.k1 = prm.k1; s.skip_k = prm.skip_k; s.W = prm.W;
    PackRegion *d_regions = nullptr;
    PackList *d_lists = nullptr;
    Slot *d_slots = nullptr;
    std::vector<void *> scratch;                                     // candidate and round scratch of every attempt
    std::vector<std::vector<PackList>> kept(regions.size());         // surviving lists, per region
    std::vector<int> todo;
    *d_slots_out = nullptr;
    *n_rounds_out = 0;
    lists.clear();
    const int n_regions = (int)regions.size();
    if (n_regions == 0) return 0;
    PD_TRY(cudaMalloc(&d_regions, sizeof(PackRegion) * n_regions));
    PD_TRY(cudaMemcpy(d_regions, regions.data(), sizeof(PackRegion) * n_regions, cudaMemcpyHostToDevice));
    count_regions_kernel<<<(n_regions + PLAN_WARPS - 1) / PLAN_WARPS, PLAN_WARPS * 32>>>(d_regions, n_regions, d_cs, s);
    count_launch();
    PD_TRY(cudaMemcpy(regions.data(), d_regions, sizeof(PackRegion) * n_regions, cudaMemcpyDeviceToHost));
    prm.split(regions, prm.split_arg);                               // sets regions[i].K
    for (int i = 0; i < n_regions; ++i)
        if (regions[i].n_in + regions[i].n_cl > 0) todo.push_back(i);
    for (int attempt = 0; !todo.empty(); ++attempt) {
        // lists of this attempt: K shares per region, candidate and round scratch by prefix sums
        std::vector<PackList> cur;
        long long cand = 0, tmp_rounds = 0;
        for (int i : todo) {
            const PackRegion &r = regions[i];
            for (int kk = 0; kk < r.K; ++kk) {
                PackList L;
                std::memset(&L, 0, sizeof(L));
                L.region = i; L.kk = kk; L.K = r.K;
                L.n = ((r.n_in > kk) ? (r.n_in - kk + r.K - 1) / r.K : 0) + ((r.n_cl > kk) ? (r.n_cl - kk + r.K - 1) / r.K : 0);
                L.cand_begin = cand; cand += L.n;
                L.round_cap = L.n / 10 + 24;                     // typical: n / 28 rounds
                L.tmp_round_begin = tmp_rounds; tmp_rounds += L.round_cap;
                cur.push_back(L);
            }
        }
        const int n_cur = (int)cur.size();
        Slot *d_cand = nullptr, *d_tmp = nullptr;
        PD_TRY(cudaMalloc(&d_cand, sizeof(Slot) * (size_t)std::max<long long>(cand, 1)));
        scratch.push_back(d_cand);
        PD_TRY(cudaMalloc(&d_tmp, sizeof(Slot) * 32 * (size_t)std::max<long long>(tmp_rounds, 1)));
        scratch.push_back(d_tmp);
        cudaFree(d_lists); d_lists = nullptr;
        PD_TRY(cudaMalloc(&d_lists, sizeof(PackList) * n_cur));
        PD_TRY(cudaMemcpy(d_lists, cur.data(), sizeof(PackList) * n_cur, cudaMemcpyHostToDevice));
        PD_TRY(cudaMemcpy(d_regions, regions.data(), sizeof(PackRegion) * n_regions, cudaMemcpyHostToDevice));
        fill_pack_kernel<<<n_cur, 32>>>(d_lists, d_regions, d_cs, s, d_cand, d_tmp, prm.pitch, prm.disjoint ? 1 : 0);
        count_launch();
        PD_TRY(cudaMemcpy(cur.data(), d_lists, sizeof(PackList) * n_cur, cudaMemcpyDeviceToHost));
        for (PackList &L : cur) {
            if (L.overflow) { rc = -2; goto done; }              // the caller falls back to the host builder
            L.src = d_tmp + (size_t)L.tmp_round_begin * 32;
        }
        std::vector<int> again;
        if (prm.redo) prm.redo(regions, cur, attempt, prm.split_arg, again);
        std::vector<char> redo_flag(n_regions, 0);
        for (int i : again) redo_flag[i] = 1;
        for (const PackList &L : cur)
            if (!redo_flag[L.region]) kept[L.region].push_back(L);
        todo = again;
    }
    {
        long long rounds = 0;
        for (int i = 0; i < n_regions; ++i)
            for (PackList &L : kept[i]) { L.round_begin = rounds; rounds += L.n_rounds; lists.push_back(L); }
        const int n_lists = (int)lists.size();
        if (n_lists == 0) goto done;
        cudaFree(d_lists); d_lists = nullptr;
        PD_TRY(cudaMalloc(&d_lists, sizeof(PackList) * n_lists));
        PD_TRY(cudaMemcpy(d_lists, lists.data(), sizeof(PackList) * n_lists, cudaMemcpyHostToDevice));
        PD_TRY(cudaMalloc(&d_slots, sizeof(Slot) * 32 * (size_t)std::max<long long>(rounds, 1)));
        compact_rounds_kernel<<<n_lists, 256>>>(d_lists, n_lists, d_slots);
        count_launch();
        PD_TRY(cudaDeviceSynchronize());
        *n_rounds_out = rounds;
        *d_slots_out = d_slots;
        d_slots = nullptr;
    }
done:
    cudaFree(d_regions); cudaFree(d_lists); cudaFree(d_slots);
    for (void *q : scratch) cudaFree(q);
    return rc;
}

// ---- both schedules of one plan half ---------------------------------------------------------------
static inline long long posmod_ll(long long v, long long m) { const long long r = v % m; return r < 0 ? r + m : r; }

struct ScatterSplitArg { int n_workers; int round_max; const std::vector<int> *k_min; const Geometry *g; bool half; };
static void scatter_split(std::vector<PackRegion> &regions, void *argp)
{
    ScatterSplitArg *arg = static_cast<ScatterSplitArg *>(argp);
    long long est = 0;
    for (const PackRegion &r : regions) est += (r.n_in + r.n_cl + 27) / 28;
    arg->round_max = scatter_round_limit(*arg->g, arg->half, est, arg->n_workers);
    // host rule (plan_host.cpp): a tile's samples are dealt to K CTAs when one warp would run more
    // than round_max rounds at ~24 samples per round
    for (PackRegion &r : regions) {
        const long long cnt = (long long)r.n_in + r.n_cl, per = 24LL * arg->round_max;
        r.K = (int)std::max<long long>(1, (cnt + per - 1) / per);
        // lanes of a round on one base row sit at least W columns apart: ~10 per row of a 64-wide tile
        r.K = std::max(r.K, (r.max_row + 10 * arg->round_max - 1) / (10 * arg->round_max));
    }
    if (arg->k_min)
        for (size_t i = 0; i < regions.size() && i < arg->k_min->size(); ++i) regions[i].K = std::max(regions[i].K, (*arg->k_min)[i]);
}
// host rule: a tile whose longest share runs more than round_max rounds is dealt to more CTAs
static void scatter_redo(std::vector<PackRegion> &regions, const std::vector<PackList> &cur, int attempt, void *argp,
                         std::vector<int> &again)
{
    ScatterSplitArg *arg = static_cast<ScatterSplitArg *>(argp);
    if (attempt >= 6) return;
    std::vector<int> mr(regions.size(), 0);
    for (const PackList &L : cur) mr[L.region] = std::max(mr[L.region], L.n_rounds);
    for (size_t i = 0; i < regions.size(); ++i)
        if (mr[i] > arg->round_max - arg->round_max / 10) {      // the longest share sets the launch's critical path
            regions[i].K = (int)std::ceil(regions[i].K * (double)mr[i] / arg->round_max * 1.15) + (attempt > 2);
            again.push_back((int)i);
        }
}
static void no_split(std::vector<PackRegion> &regions, void *)
{
    for (PackRegion &r : regions) r.K = 1;
}

int build_schedules_device(const Geometry &g, const double2 *d_cs, bool half, int n_workers, Schedules &out,
                           Slot **d_gather_slots, long long *n_gather_rounds,
                           Slot **d_scatter_slots, long long *n_scatter_rounds)
{
    out = Schedules();
    out.half = half;
    *d_gather_slots = *d_scatter_slots = nullptr;
    const int G = g.G, KW = g.W, KH = KW - 1;
    int gk0, gk1, sk1;
    sample_ranges(g, half, gk0, gk1, sk1);
    DevicePackParams prm;
    prm.n_angles = g.n_angles; prm.n_det = g.n_det; prm.G = G; prm.W = KW;
    std::vector<PackRegion> regions;
    std::vector<PackList> lists;

    // ---- gather: tiles of GT_X x GT_Y base cells (rows counted from yorg on the half schedule)
    {
        const int yorg = half ? (int)posmod_ll(G / 2 - KW / 2, G) : 0;
        for (int ry0 = 0; ry0 < G; ry0 += GT_Y)
            for (int rx0 = 0; rx0 < G; rx0 += GT_X) {
                PackRegion r;
                std::memset(&r, 0, sizeof(r));
                r.rx0 = rx0; r.ry0 = ry0; r.rw = std::min(GT_X, G - rx0); r.rh = std::min(GT_Y, G - ry0);
                r.lo = 0; r.oy = yorg; r.K = 1;
                regions.push_back(r);
            }
        prm.k0 = gk0; prm.k1 = gk1; prm.skip_k = -1; prm.pitch = gt_pitch(KW); prm.disjoint = false;
        prm.split = no_split; prm.redo = nullptr; prm.split_arg = nullptr;
        int rc = device_pack(d_cs, prm, regions, lists, d_gather_slots, n_gather_rounds);
        if (rc) return rc;
        for (const PackList &L : lists) {
            const PackRegion &r = regions[L.region];
            out.gather_filled += L.filled;
            for (int q = 0; q < L.n_rounds; q += GATHER_ROUND_CAP) {
                GatherCta c;
                c.tx0 = r.rx0; c.ty0 = (int)posmod_ll((long long)yorg + r.ry0, G);
                c.round_begin = (int)L.round_begin + q;
                c.round_count = std::min(GATHER_ROUND_CAP, L.n_rounds - q);
                out.gather_ctas.push_back(c);
            }
        }
        finish_gather(out, n_workers);
    }

    // ---- scatter: one list per (tile, share); tiles that are split or hold the centre window are merge jobs
    {
        std::vector<TileRect> tiles;
        scatter_tile_rects(g, half, tiles);
        regions.clear();
        for (const TileRect &t : tiles) {
            PackRegion r;
            std::memset(&r, 0, sizeof(r));
            r.rx0 = t.rx0; r.ry0 = t.ry0; r.rw = t.rw; r.rh = t.rh; r.lo = KH; r.oy = 0; r.K = 1;
            regions.push_back(r);
        }
        // Where samples pile up on few base cells (the centre) a share needs more rounds than its
        // sample count suggests: like the host builder, such a tile is dealt to more CTAs and packed again.
        ScatterSplitArg arg{n_workers, SCATTER_ROUND_MAX, nullptr, &g, half};
        prm.k0 = 0; prm.k1 = sk1; prm.skip_k = g.n_det / 2; prm.pitch = ACC_PITCH; prm.disjoint = true;
        prm.split = scatter_split; prm.redo = scatter_redo; prm.split_arg = &arg;
        {
            int rc = device_pack(d_cs, prm, regions, lists, d_scatter_slots, n_scatter_rounds);
            if (rc) { cudaFree(*d_gather_slots); *d_gather_slots = nullptr; return rc; }
        }
        // tiles without a sample are still written (zeros): they get one list-less CTA each
        std::vector<int> first_list(regions.size(), -1);
        for (size_t i = 0; i < lists.size(); ++i)
            if (first_list[lists[i].region] < 0) first_list[lists[i].region] = (int)i;
        struct Pending { ScatterCta cta; long long work; };
        std::vector<Pending> ctas;
        for (size_t ri = 0; ri < regions.size(); ++ri) {
            const PackRegion &r = regions[ri];
            bool has_dc = false;
            for (int uy = (half ? 0 : -KW / 2); uy <= KW / 2; ++uy)
                for (int ux = -KW / 2; ux <= KW / 2; ++ux) {
                    const int cx = G / 2 + ux, cy = G / 2 + uy;
                    has_dc = has_dc || (cx >= r.rx0 && cx < r.rx0 + r.rw && cy >= r.ry0 && cy < r.ry0 + r.rh);
                }
            const int K = (first_list[ri] < 0) ? 1 : r.K;
            int first_slot = -1, job = -1;
            if (K > 1 || has_dc) {
                first_slot = out.n_partial_slots;
                out.n_partial_slots += K;
                job = (int)out.merge_jobs.size();
                out.merge_jobs.push_back(MergeJob{r.rx0, r.ry0, r.rw, r.rh, first_slot, K, K + (has_dc ? 1 : 0), 0});
                if (has_dc) out.dc_jobs.push_back(job);
            }
            for (int kk = 0; kk < K; ++kk) {
                Pending p;
                std::memset(&p.cta, 0, sizeof(p.cta));
                p.cta.rx0 = r.rx0; p.cta.ry0 = r.ry0; p.cta.rw = r.rw; p.cta.rh = r.rh;
                p.cta.partial_slot = (job >= 0) ? first_slot + kk : -1;
                p.cta.job = job;
                ScatterItem &it = p.cta.items[0];
                it.sx0 = 0; it.sy0 = 0; it.sw = r.rw; it.sh = r.rh;
                if (first_list[ri] >= 0) {
                    const PackList &L = lists[first_list[ri] + kk];
                    it.round_begin = (int)L.round_begin; it.round_count = L.n_rounds; it.fast_count = L.n_fast;
                    out.scatter_filled += L.filled;
                }
                p.work = it.round_count;
                ctas.push_back(p);
            }
        }
        std::stable_sort(ctas.begin(), ctas.end(), [](const Pending &x, const Pending &y) { return x.work > y.work; });
        for (const Pending &p : ctas) out.scatter_ctas.push_back(p.cta);
    }
    return 0;
}

}  // namespace radon

// ---- density compensation of the inverse Radon transform on the device ---------------
// D(x_i, y_i) = scale / sum_j K(x_i - x_j, y_i - y_j), the sum over ALL polar samples, K = phi(dx) phi(dy).
// One thread per sample i.  Its neighbours are found from the geometry: only radial lines that pass
// within W/2 sqrt 2 of the sample can hold one (all lines near the centre, a window of angles
// further out), and on a line the samples inside the W x W box are an interval of j (as in
// for_candidates).  phi is evaluated in fp64 from the series of I0; the terms are added in a fixed
// order.  Checked against the host table (build_density) to fp32 round-off.
namespace radon {

__device__ __forceinline__ double i0_series(double z)
{
    const double q = 0.25 * z * z;
    double term = 1.0, sum = 1.0;
    for (int m = 1; m < 200; ++m) {
        term *= q / ((double)m * (double)m);
        sum += term;
        if (term < 1e-17 * sum) break;
    }
    return sum;
}

__device__ __forceinline__ double kb_phi_dev(double u, double beta, double inv_i0b, int KW)
{
    const double t = 2.0 * u / (double)KW, arg = 1.0 - t * t;
    if (arg < 0.0) return (arg > -1e-12) ? inv_i0b : 0.0;       // |u| == W/2 up to rounding
    return i0_series(beta * sqrt(arg)) * inv_i0b;
}

__global__ void __launch_bounds__(128)
density_kernel(float *__restrict__ D, const double2 *__restrict__ cs, int n_angles, int n_det, int KW, double beta,
               double inv_i0b, double scale)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)n_angles * n_det) return;
    const int a = (int)(i / n_det), k = (int)(i - (long long)a * n_det), cd = n_det / 2;
    const double2 d = cs[a];
    const double kx = (double)(k - cd) * d.x, ky = (double)(k - cd) * d.y, hw = 0.5 * KW;
    const double r = sqrt(kx * kx + ky * ky);
    // lines that can come within hw * sqrt(2) of the sample: |sin(theta' - theta)| <= hw sqrt 2 / r
    int win = n_angles;                                         // offsets -win .. +win (all lines when >= n_angles / 2)
    const double reach = hw * 1.4142135623730951 + 1e-6;
    if (r > reach) win = (int)ceil(asin(reach / r) / (3.14159265358979323846 / (double)n_angles)) + 1;
    const bool all = 2 * win + 1 >= n_angles;
    const int o_lo = all ? 0 : -win, o_hi = all ? n_angles - 1 : win;
    double sum = 0.0;
    for (int o = o_lo; o <= o_hi; ++o) {
        int a2 = all ? o : (a + o) % n_angles;
        if (a2 < 0) a2 += n_angles;
        const double2 e = cs[a2];
        // j e in [kappa - hw, kappa + hw] on both axes: an interval of j
        double lo = -(double)cd - 0.5, hi = (double)(n_det - 1 - cd) + 0.5;
        if (fabs(e.x) > 1e-12) { const double u = (kx - hw) / e.x, v = (kx + hw) / e.x; lo = fmax(lo, fmin(u, v) - 1e-6); hi = fmin(hi, fmax(u, v) + 1e-6); }
        else if (fabs(kx) > hw + 1e-9) continue;
        if (fabs(e.y) > 1e-12) { const double u = (ky - hw) / e.y, v = (ky + hw) / e.y; lo = fmax(lo, fmin(u, v) - 1e-6); hi = fmin(hi, fmax(u, v) + 1e-6); }
        else if (fabs(ky) > hw + 1e-9) continue;
        for (int j = (int)ceil(lo); j <= (int)floor(hi); ++j) {
            const double px = kb_phi_dev(kx - (double)j * e.x, beta, inv_i0b, KW);
            if (px != 0.0) sum += px * kb_phi_dev(ky - (double)j * e.y, beta, inv_i0b, KW);
        }
    }
    D[i] = (float)(scale / sum);
}

// even n_det: the Hermitian-half scatter needs the mean weight of every +-j pair
__global__ void density_pair_mean_kernel(float *__restrict__ D, int n_angles, int n_det)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int half = n_det / 2 - 1;                             // pairs k = 1 .. n/2 - 1 with n - k
    if (half <= 0 || i >= (long long)n_angles * half) return;
    const int a = (int)(i / half), k = 1 + (int)(i - (long long)a * half);
    float *row = D + (size_t)a * n_det;
    const float m = 0.5f * (row[k] + row[n_det - k]);
    row[k] = m; row[n_det - k] = m;
}

int launch_density(const double2 *d_cs, int n_angles, int n_det, int W, double beta, double inv_i0b, double scale,
                   float *d_D, cudaStream_t st)
{
    const long long M = (long long)n_angles * n_det;
    density_kernel<<<(unsigned)((M + 127) / 128), 128, 0, st>>>(d_D, d_cs, n_angles, n_det, W, beta, inv_i0b, scale);
    count_launch();
    return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

int launch_density_pair_mean(float *d_D, int n_angles, int n_det, cudaStream_t st)
{
    const long long n = (long long)n_angles * (n_det / 2 - 1);
    if ((n_det & 1) || n <= 0) return 0;
    density_pair_mean_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d_D, n_angles, n_det);
    count_launch();
    return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace radon
