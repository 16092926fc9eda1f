// radon_internal.h -- data structures shared by the host-side plan builder and the
// CUDA kernels of libradon_b200.  Not part of the public ABI (include/radon.h is).
#pragma once
#include <cstdint>
#include <vector>

namespace radon {

// ---- compile-time configuration -------------------------------------------------
// Kaiser-Bessel widths this build carries: the gridding kernels are instantiated for each (even
// widths: the polynomial pieces pair up), the host code takes W at run time.  A footprint reaches
// base .. base + W - 1 ("halo" W - 1).
constexpr int KW_MAX = 8;
inline bool kw_supported(int W) { return W == 4 || W == 6 || W == 8; }
#define RADON_FOR_W(Wrt, BODY)                        \
    switch (Wrt) {                                    \
    case 4: { constexpr int WW = 4; BODY } break;     \
    case 6: { constexpr int WW = 6; BODY } break;     \
    case 8: { constexpr int WW = 8; BODY } break;     \
    default: break;                                   \
    }
// Kaiser-Bessel weights: ONE polynomial piece per tap (degree KB_DEG in z = 2*delta - 1, fitted
// in fp64 at plan time, max error ~7e-8), passed to the kernels in the constant bank -- a lookup
// table whose rows are polynomial pieces, read as broadcast operands, so it costs neither
// shared-memory bandwidth nor bank conflicts.  north_star's shared-memory LUT with linear
// interpolation was built and measured against it (profiles/r02_kb_lut_ab.md: 256 rows per grid
// unit cost 3e-6 of the 1e-5 budget, 1024 rows 48 KB of shared memory per CTA, and either makes
// the gather 56 % slower); the polynomial pieces are what the library ships.
constexpr int KB_DEG = 7;
constexpr int KB_HALF = (KB_DEG + 1) / 2;   // coefficients of the even / odd part
struct KbPoly {                       // tap l: E_l(z^2) + z O_l(z^2); tap W-1-l: E_l - z O_l
    float e[KW_MAX / 2][KB_HALF];
    float o[KW_MAX / 2][KB_HALF];
};
#ifdef __CUDACC__
#define RADON_HD __host__ __device__ __forceinline__
#else
#define RADON_HD inline
#endif
// w[l] = phi(delta - W/2 + l), l = 0..W-1, delta in [0,1]: Horner in z^2 on the even and odd
// parts.  In the kernels kp sits in the parameter constant bank, so its entries are FFMA
// operands, not loads.  Host-callable for the CPU-side unit test.
template <int W>
RADON_HD void kb_poly_weights(const KbPoly &kp, float delta, float (&w)[W])
{
    const float z = 2.f * delta - 1.f, z2 = z * z;
#ifdef __CUDACC__
#pragma unroll
#endif
    for (int l = 0; l < W / 2; ++l) {
        float e = kp.e[l][KB_HALF - 1], o = kp.o[l][KB_HALF - 1];
#ifdef __CUDACC__
#pragma unroll
#endif
        for (int h = KB_HALF - 2; h >= 0; --h) {
            e = e * z2 + kp.e[l][h];
            o = o * z2 + kp.o[l][h];
        }
        w[l] = e + z * o;
        w[W - 1 - l] = e - z * o;
    }
}
// Gather (inverse gridding): a work item is a GT_X x GT_Y tile of the grid (+halo), staged by
// one bulk copy per tile row.  Wide, flat tiles: the copy engine spends ~65 cycles per copy
// whatever its size (measured: 1 KB copies reach 4.5 TB/s over 148 SMs, >= 2 KB copies the HBM
// rate), so a row of 3 KB is worth the larger halo (21/16 rows); three tiles in flight per CTA
// (measured at config 4, bare kernel: 128 x 64 x 3 stages 62 us, 512 x 16 x 2 55 us, 384 x 16 x 3 49 us).
#ifndef RADON_GT_X
#define RADON_GT_X 384
#define RADON_GT_Y 16
#define RADON_GSTAGES 3
#endif
constexpr int GT_X = RADON_GT_X, GT_Y = RADON_GT_Y;
constexpr int gt_pitch(int W) { return GT_X + W; }       // complex per smem row (tile + halo W - 1, + 1): 16-byte multiple for the bulk copies
constexpr int gt_rows(int W) { return GT_Y + W - 1; }    // rows staged per tile (21 at W = 6)
constexpr int GT_ROWS_MAX = gt_rows(KW_MAX);
#ifndef RADON_GWARPS
#define RADON_GWARPS 24
#endif
constexpr int GATHER_WARPS = RADON_GWARPS;      // consumer warps of the persistent gather CTA (+1 producer warp)
constexpr int GATHER_STAGES = RADON_GSTAGES;   // tiles in flight per CTA (gt_rows x gt_pitch x 8 B = 65.5 KB each at W = 6)
#ifndef RADON_GCOST
#define RADON_GCOST 16
#endif
constexpr int GATHER_ITEM_COST = RADON_GCOST;  // load balancing: an item costs its rounds + this (tile staging)
#ifndef RADON_GCAP
#define RADON_GCAP 64
#endif
constexpr int GATHER_ROUND_CAP = RADON_GCAP;  // rounds (of 32 samples) per CTA; heavier tiles get more CTAs

// Scatter (gridding): a CTA accumulates one SR_X x SR_Y output rectangle in shared memory;
// each of its SQ_X x SQ_Y warps owns one ST_X x ST_Y tile of it and processes every sample whose
// footprint intersects that tile, taps clipped to the tile (so warps never share a cell, and the
// accumulator needs no margins).  Default: ONE warp per CTA (SQ = 1 x 1, 64 x 32 tile, 17 KB,
// twelve CTAs per multiprocessor): no CTA barrier, and the fixed cost of a tile (descriptor, first
// slots, first sample values: three dependent global loads; the flush) overlaps the accumulation
// of eleven independent warps.  Measured at config 4 against four warps per 128 x 64 rectangle at
// three CTAs per multiprocessor: bare 92.7 -> 89.0 us, A2 stage 58.1 -> 56.9 us, 32-slice batch
// 185.6 -> 180.4 us per pair.  Grids of ST_Y_TALL_MIN_G and more use tiles of ST_Y_TALL rows (below).
#ifndef RADON_SC_FAST
#define RADON_SC_FAST 1               // unclipped footprints first, run without tap predicates
#endif
#ifndef RADON_SC_STEP_ROWS
#define RADON_SC_STEP_ROWS 1          // footprint rows a lane adds between two warp barriers (fast rounds)
#endif
constexpr int SC_STEP_ROWS = RADON_SC_STEP_ROWS;
static_assert(SC_STEP_ROWS == 1 || SC_STEP_ROWS == 2 || SC_STEP_ROWS == 3, "6 rows in steps of 1, 2 or 3");
#ifndef RADON_ST_X
#define RADON_ST_X 64
#define RADON_ST_Y 32
#define RADON_SQ_X 1
#define RADON_SQ_Y 1
#define RADON_SC_CTAS 12
#endif
constexpr int ST_X = RADON_ST_X, ST_Y = RADON_ST_Y;
constexpr int SQ_X = RADON_SQ_X, SQ_Y = RADON_SQ_Y;   // quadrants per rectangle
constexpr int SR_X = SQ_X * ST_X, SR_Y = SQ_Y * ST_Y; // CTA output rectangle
constexpr int SCATTER_ITEMS = SQ_X * SQ_Y;            // warps per CTA
constexpr int ACC_PITCH = SR_X + 2;   // 130 complex per accumulator row (16-byte multiple, != 0 mod 16)
// Tile height is a property of the plan: ST_Y rows, or ST_Y_TALL on large grids (Geometry::st_y), where the
// scatter is bound by shared-memory bandwidth, not latency: eight to ten warps per multiprocessor fill
// the pipe, and taller tiles list fewer footprints twice and pay fewer prologues.
#ifndef RADON_ST_Y_TALL
#define RADON_ST_Y_TALL 40
#define RADON_SC_CTAS_TALL 10
#endif
constexpr int ST_Y_TALL = (SCATTER_ITEMS == 1) ? RADON_ST_Y_TALL : ST_Y;
#ifndef RADON_ST_Y_TALL_MIN_G
#define RADON_ST_Y_TALL_MIN_G 4096
#endif
constexpr int ST_Y_TALL_MIN_G = RADON_ST_Y_TALL_MIN_G;               // grids at least this wide get the tall tiles
constexpr int SCATTER_CTAS_PER_SM_TALL = RADON_SC_CTAS_TALL;   // 10 x 21 KB of accumulators
constexpr int SB_W_MAX = ST_X + KW_MAX - 1, SB_H_MAX = ST_Y_TALL + KW_MAX - 1;   // range of biased base coordinates in a tile (ST + W - 1)
constexpr int SCATTER_ROUND_MAX = 96; // rounds per warp before a tile's samples are split over CTAs: upper and
#ifndef RADON_SC_RMIN
#define RADON_SC_RMIN 12
#endif
#define RADON_SC_RFAC_FULL_DEFAULT 1.8
#ifndef RADON_SC_RFAC_FULL
#define RADON_SC_RFAC_FULL RADON_SC_RFAC_FULL_DEFAULT
#endif
#ifndef RADON_SC_RFAC_TALL_FULL
#define RADON_SC_RFAC_TALL_FULL 1.2      // the full-grid schedule of the tall tiles (twice the rounds per warp of the half one)
#endif
#ifndef RADON_SC_RFAC_TALL
#define RADON_SC_RFAC_TALL 1.5           // the same for the tall tiles, Hermitian-half schedule (1.2-1.8 measured)
#endif
#ifndef RADON_SC_RFAC
#define RADON_SC_RFAC 1.8                // split limit = RFAC x the mean rounds per resident warp (0.7-1.8 measured)
#endif
constexpr int SCATTER_ROUND_MIN = RADON_SC_RMIN;  // lower limit (12: best over configs 1-3 and the paper's shape, 8..24 measured); the builder
                                      // picks 1.8 x the mean rounds per resident warp
constexpr int SCATTER_CTAS_PER_SM = RADON_SC_CTAS;

// One lane's work in one round: which polar sample, and where its W x W footprint
// starts inside the staged tile (gather) or the warp-private accumulator (scatter).
struct Slot {
    uint32_t ak;    // (a << 16) | k ; 0xFFFFFFFF = idle lane
    uint32_t lxy;   // lx0 | (ly0 << 16)
};
constexpr uint32_t SLOT_EMPTY = 0xFFFFFFFFu;

struct GatherCta {              // one work item of the gather: a staged tile and some of its rounds
    int tx0, ty0;               // tile origin (cells, centred layout)
    int round_begin, round_count;
};

struct ScatterItem {            // one warp: quadrant (relative to the rectangle) and its rounds
    int sx0, sy0, sw, sh;       // slot coordinates are relative to (sx0 - (W-1), sy0 - (W-1))
    int round_begin, round_count;
    int fast_count;             // the first fast_count rounds hold only footprints wholly inside the quadrant
    int pad;
};

struct ScatterCta {
    int rx0, ry0, rw, rh;       // output rectangle (cells this CTA, alone, writes)
    int partial_slot;           // -1: write the grid; >= 0: write this scratch slot
    int job;                    // merge job the partial rectangle belongs to (-1: none)
    int pad1, pad2;
    ScatterItem items[SCATTER_ITEMS];
};

// A rectangle whose samples are split over several CTAs (polar sampling is ~1/r dense), or
// that holds cells of the centre window the summed j = 0 samples are added to: every CTA of
// the job writes its partial rectangle to a scratch slot and takes a ticket; whoever draws the
// last ticket sums the slots IN SLOT ORDER (bitwise reproducible whatever the arrival order).
struct MergeJob {
    int rx0, ry0, rw, rh;
    int first_slot, n_slots;
    int expected;               // tickets: n_slots, + 1 when the j = 0 sum (dc) takes part
    int pad;
};
constexpr int MAX_DC_JOBS = 4;  // the (W+1)^2 centre window touches at most 2 x 2 rectangles

// ---- host-side geometry + schedules ----------------------------------------------
struct Geometry {
    int N = 0, G = 0, n_angles = 0, n_det = 0, W = 6;
    double sigma = 2.0;
    int st_y = ST_Y;            // rows of a scatter tile (ST_Y or ST_Y_TALL)
    int sr_y() const { return SQ_Y * st_y; }                                  // rows of a CTA's rectangle
    int scatter_ctas_per_sm() const { return st_y == ST_Y ? SCATTER_CTAS_PER_SM : SCATTER_CTAS_PER_SM_TALL; }
    double scatter_rfac(bool half) const { return st_y == ST_Y ? (half ? RADON_SC_RFAC : RADON_SC_RFAC_FULL) : (half ? RADON_SC_RFAC_TALL : RADON_SC_RFAC_TALL_FULL); }
    std::vector<double> cs;     // per angle: (G/n) cos(theta_a), (G/n) sin(theta_a)

    void init(int N_, int n_angles_, int n_det_, double sigma_, int W_);
    // Base cell (centred layout, may lie in [-W/2, G - W/2]) of sample (a, k):
    // x0 = ceil(G/2 + kappa_x - W/2).  Bit-identical to the device code (same fma).
    void base(int a, int k, int &x0, int &y0) const;
};

struct Schedules {
    std::vector<Slot> gather_slots;         // 32 per round
    std::vector<GatherCta> gather_ctas;     // work items, grouped by persistent CTA
    std::vector<int> gather_worker_begin;   // persistent CTA w owns items [begin[w], begin[w+1])
    std::vector<Slot> scatter_slots;
    std::vector<ScatterCta> scatter_ctas;
    std::vector<MergeJob> merge_jobs;
    std::vector<int> dc_jobs;               // merge jobs whose rectangle holds cells of the centre window
    int n_partial_slots = 0;
    bool half = false;
    long long gather_filled = 0, scatter_filled = 0;
};

// half == false: every sample, the whole grid (arbitrary complex data: the test hooks).
// half == true:  Hermitian half for real images / sinograms (radon_forward, radon_adjoint).
// n_workers: persistent CTAs of the gather (one per multiprocessor).
void build_schedules(const Geometry &g, Schedules &out, bool half, int n_workers = 148);
// pieces of the builder shared with the device-side builder (plan_device.cu)
struct TileRect { int rx0, ry0, rw, rh; };
void scatter_tile_rects(const Geometry &g, bool half, std::vector<TileRect> &tiles);   // tiles the scatter writes
void sample_ranges(const Geometry &g, bool half, int &gather_k0, int &gather_k1, int &scatter_k1);
int scatter_round_limit(const Geometry &g, bool half, long long est_rounds, int n_workers);    // rounds per warp before a tile is split
void finish_gather(Schedules &out, int n_workers);               // gather items -> persistent CTAs
// Returns the number of violated invariants (0 = schedules are valid).
long long check_schedules(const Geometry &g, const Schedules &s);

// ---- host-side tables (all derived in fp64, stored fp32) -------------------------
double kb_beta(int W, double sigma);
double kb_i0(double z);
void build_kb_poly(int W, double sigma, KbPoly &kp);                            // Chebyshev fit, fp64
void build_deapod(int N, int G, int W, double sigma, std::vector<float> &d);   // N floats
void build_twiddles(int L, std::vector<float> &tw);                            // L x (cos, -sin)
// Bluestein / centred-DFT tables for length n, FFT length L (power of two >= 2n-1, or
// L == n when n is a power of two: then hf is empty and a/b are the centring phases).
void build_chirp(int n, int L, std::vector<float> &a, std::vector<float> &b, std::vector<float> &hf);
int next_pow2(int v);
// Sinogram filter: orthonormal discrete polynomials q_0 .. q_order on n
// equispaced points, fp64 Gram-Schmidt (twice) on the monomials of t in [-1, 1], stored fp32 as
// q[s * FILTER_MAXQ + d] (rows beyond the order are zero).
constexpr int FILTER_MAXQ = 8;              // orders 0 .. 7
constexpr int FILTER_FUSED_Q = 4;           // the fused kernels (proj.cu) carry orders 0 .. 3
void build_filter_basis(int n, int order, std::vector<float> &q);
// Density compensation of the inverse Radon transform: D_i = 1 / sum_j K(x_i - x_j, y_i - y_j)
// over all polar samples, times the quadrature scale n phihat(0)^2 / G^2; fp64, stored fp32.
void build_density(const Geometry &g, std::vector<float> &D, double *scale_out);

// ---- the paper's own gridding design, kept as a measured comparison ----------
// "The load balancing algorithm starts by considering one bin containing all the points, and
// recursively divides the most computationally intensive bin into four equally sized bins (the
// computational cost is estimated as the number of samples times the number of grid points in
// each bin) ... one thread block per bin."  A bin lists every sample image whose W x W footprint
// touches it (a sample near a border is listed by both neighbours).
struct PaperBin {
    int x0, y0, w, h;           // cells [x0, x0 + w) x [y0, y0 + h) of the centred grid
    int first, count;           // entries [first, first + count) of the sample list
};
struct PaperBinEntry {
    uint32_t ak;                // (a << 16) | k
    int32_t shift;              // wrap image: (sx + 1) | ((sy + 1) << 2), base cell = (x0 + sx G, y0 + sy G)
};
struct PaperBins {
    std::vector<PaperBin> bins;             // heaviest first
    std::vector<PaperBinEntry> entries;
};
// n_bins_target: stop splitting once there are this many bins (or no bin can be split: side 8)
void build_paper_bins(const Geometry &g, int n_bins_target, PaperBins &out);

}  // namespace radon
