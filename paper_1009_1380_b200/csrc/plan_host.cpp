// plan_host.cpp -- host side of radon_plan_create: Fourier-slice geometry, tables and
// the plan-time gather / scatter schedules.  Pure C++ (no CUDA calls) so that it can be
// exercised on a machine without a GPU (radon_schedule_selfcheck).
//
// The schedules take the place of the paper's load-balanced bins ("recursively divides
// the most computationally intensive bin into four"): the geometry of a plan
// is fixed, so every decision the paper's kernels take at run time (which block owns which
// samples, in which order they accumulate) is taken here once:
//   * samples are binned into grid tiles by a counting sort;
//   * inside a tile they are packed into ROUNDS of 32 (one per lane of a warp) such that
//       - the lanes of each half-warp start in distinct shared-memory bank pairs, so every
//         64-bit tap access of the round is conflict free (all lanes add the same tap offset
//         to their base); lanes that would otherwise stay idle may share a bank pair with one
//         other lane (2-way conflict: one extra wavefront instead of another round), and
//       - (scatter only) no two lanes of a round touch the same cell within a row step (same
//         base row, base columns closer than W), so the warp can accumulate with plain
//         load/add/store: no atomics, and the order of every floating-point addition is
//         fixed -> bitwise reproducible;
//   * tiles whose sample count (polar sampling is ~1/r dense: PAPER.md:57's imbalance) would
//     make one block run long are split over several warps / blocks by dealing their samples
//     round-robin; partial rectangles are summed in slot order by the last CTA of the tile
//     to finish (ticket), inside the scatter launch.
#include "radon_internal.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>
#include <thread>

namespace radon {

static const double kPi = 3.14159265358979323846264338327950288;

int next_pow2(int v)
{
    int p = 1;
    while (p < v) p <<= 1;
    return p;
}

// ---------------------------------------------------------------- geometry -------
void Geometry::init(int N_, int n_angles_, int n_det_, double sigma_, int W_)
{
    N = N_; n_angles = n_angles_; n_det = n_det_; sigma = sigma_; W = W_;
    G = (int)std::llround(sigma * N);
    st_y = (G >= ST_Y_TALL_MIN_G) ? ST_Y_TALL : ST_Y;
    cs.resize(2 * (size_t)n_angles);
    const double scale = (double)G / (double)n_det;
    for (int a = 0; a < n_angles; ++a) {
        double c, s;
        if (2 * a == n_angles) { c = 0.0; s = 1.0; }         // theta = pi/2 exactly
        else {
            const double th = kPi * (double)a / (double)n_angles;
            c = std::cos(th); s = std::sin(th);
        }
        cs[2 * a] = scale * c;
        cs[2 * a + 1] = scale * s;
    }
}

void Geometry::base(int a, int k, int &x0, int &y0) const
{
    const double jj = (double)(k - n_det / 2);
    const double half = 0.5 * (double)G, hw = 0.5 * (double)W;
    const double gx = std::fma(jj, cs[2 * a], half);
    const double gy = std::fma(jj, cs[2 * a + 1], half);
    x0 = (int)std::ceil(gx - hw);
    y0 = (int)std::ceil(gy - hw);
}

// ---------------------------------------------------------------- tables ---------
double kb_i0(double z)
{
    const double q = 0.25 * z * z;
    double term = 1.0, sum = 1.0;
    for (int m = 1; m < 1000; ++m) {
        term *= q / ((double)m * (double)m);
        sum += term;
        if (term < 1e-18 * sum) break;
    }
    return sum;
}

double kb_beta(int W, double sigma)
{
    const double r = (double)W / sigma * (sigma - 0.5);
    return kPi * std::sqrt(r * r - 0.8);
}

static double kb_phi(double u, int W, double beta, double inv_i0b)
{
    const double t = 2.0 * u / (double)W;
    const double arg = 1.0 - t * t;
    if (arg < 0.0) return (arg > -1e-12) ? inv_i0b : 0.0;   // |u| == W/2 up to rounding
    return kb_i0(beta * std::sqrt(arg)) * inv_i0b;
}

// Polynomial pieces of the kernel: for tap l (l < W/2) and delta in [0,1), z = 2 delta - 1,
//   phi(delta - W/2 + l) = p_l(z),  phi(delta - W/2 + (W-1-l)) = p_l(-z)   (phi is even).
// p_l is the degree-KB_DEG truncation of the Chebyshev series of phi on the piece (64-node
// discrete cosine transform in fp64), converted to the monomial basis and split into even
// and odd parts.
void build_kb_poly(int W, double sigma, KbPoly &kp)
{
    const double beta = kb_beta(W, sigma), inv = 1.0 / kb_i0(beta);
    const int NN = 64, D = KB_DEG;
    for (int l = 0; l < W / 2; ++l) {
        double f[NN], c[D + 1];
        for (int i = 0; i < NN; ++i) {
            const double z = std::cos(kPi * (i + 0.5) / NN);
            f[i] = kb_phi(0.5 * (z + 1.0) - 0.5 * W + l, W, beta, inv);
        }
        for (int k = 0; k <= D; ++k) {
            double acc = 0.0;
            for (int i = 0; i < NN; ++i) acc += f[i] * std::cos(kPi * k * (i + 0.5) / NN);
            c[k] = (k == 0 ? 1.0 : 2.0) * acc / NN;
        }
        // Chebyshev -> monomial: T_0 = 1, T_1 = z, T_{k+1} = 2 z T_k - T_{k-1}
        double mono[D + 1] = {0}, t0[D + 1] = {0}, t1[D + 1] = {0}, t2[D + 1];
        t0[0] = 1.0; t1[1] = 1.0;
        for (int i = 0; i <= D; ++i) mono[i] += c[0] * t0[i] + c[1] * t1[i];
        for (int k = 2; k <= D; ++k) {
            for (int i = 0; i <= D; ++i) t2[i] = (i > 0 ? 2.0 * t1[i - 1] : 0.0) - t0[i];
            for (int i = 0; i <= D; ++i) { mono[i] += c[k] * t2[i]; t0[i] = t1[i]; t1[i] = t2[i]; }
        }
        for (int h = 0; h < KB_HALF; ++h) {
            kp.e[l][h] = (float)mono[2 * h];
            kp.o[l][h] = (2 * h + 1 <= D) ? (float)mono[2 * h + 1] : 0.f;
        }
    }
}

void build_deapod(int N, int G, int W, double sigma, std::vector<float> &d)
{
    const double beta = kb_beta(W, sigma), scale = (double)W / kb_i0(beta);
    d.resize(N);
    for (int i = 0; i < N; ++i) {
        const double xi = (double)(i - N / 2) / (double)G;
        const double a = kPi * W * xi, r = beta * beta - a * a;
        double ph;
        if (r > 0) { const double q = std::sqrt(r); ph = scale * std::sinh(q) / q; }
        else if (r < 0) { const double q = std::sqrt(-r); ph = scale * std::sin(q) / q; }
        else ph = scale;
        d[i] = (float)(1.0 / ph);
    }
}

// ---------------------------------------------------------------- density --------
// PAPER.md:89.  Plan-time constant (like the de-apodisation vector): derived on the host in
// fp64 on first use of radon_inverse.  Samples are bucketed by grid cell; the kernel comes from
// a fine table (8192 entries per grid unit, linear interpolation: error ~2e-9, far below the
// fp32 the weights are stored in), the sum over a sample's neighbours runs on all host threads.
void build_density(const Geometry &g, std::vector<float> &D, double *scale_out)
{
    const int G = g.G, W = g.W, n = g.n_det;
    const long long M = (long long)g.n_angles * n;
    const double beta = kb_beta(W, g.sigma), inv = 1.0 / kb_i0(beta);
    constexpr int TS = 8192;
    const int TL = (W / 2) * TS;
    std::vector<double> tab((size_t)TL + 2);
    for (int i = 0; i <= TL + 1; ++i) tab[i] = kb_phi(std::min((double)i / TS, 0.5 * W), W, beta, inv);
    tab[TL + 1] = 0.0;
    auto phi = [&](double u) {
        const double t = std::fabs(u) * TS;
        if (t > (double)TL) return 0.0;
        const int i = (int)t;
        return tab[i] + (t - i) * (tab[i + 1] - tab[i]);
    };
    std::vector<double> kx((size_t)M), ky((size_t)M);
    for (int a = 0; a < g.n_angles; ++a)
        for (int k = 0; k < n; ++k) {
            const double jj = (double)(k - n / 2);
            kx[(size_t)a * n + k] = jj * g.cs[2 * a];
            ky[(size_t)a * n + k] = jj * g.cs[2 * a + 1];
        }
    const int B = G + 3, R = W / 2 + 1;
    std::vector<long long> start((size_t)B * B + 1, 0), order((size_t)M);
    std::vector<int> cell((size_t)M);
    for (long long m = 0; m < M; ++m) {
        const int cx = (int)std::floor(kx[m]) + G / 2 + 1, cy = (int)std::floor(ky[m]) + G / 2 + 1;
        cell[m] = cy * B + cx;
        ++start[cell[m] + 1];
    }
    for (size_t c = 0; c < (size_t)B * B; ++c) start[c + 1] += start[c];
    {
        std::vector<long long> fill(start.begin(), start.end() - 1);
        for (long long m = 0; m < M; ++m) order[fill[cell[m]]++] = m;
    }
    // phihat(0) = W/I0(beta) * sinh(beta)/beta: the integral of the kernel
    const double ph0 = (double)W * inv * std::sinh(beta) / beta;
    const double scale = (double)n * ph0 * ph0 / ((double)G * (double)G);
    if (scale_out) *scale_out = scale;
    D.resize((size_t)M);
    auto work = [&](long long lo, long long hi) {
        for (long long i = lo; i < hi; ++i) {
            const int cx = cell[i] % B, cy = cell[i] / B;
            double s = 0.0;
            for (int y = std::max(cy - R, 0); y <= std::min(cy + R, B - 1); ++y)
                for (int x = std::max(cx - R, 0); x <= std::min(cx + R, B - 1); ++x)
                    for (long long q = start[(size_t)y * B + x]; q < start[(size_t)y * B + x + 1]; ++q) {
                        const long long j = order[q];
                        const double px = phi(kx[i] - kx[j]);
                        if (px != 0.0) s += px * phi(ky[i] - ky[j]);
                    }
            D[i] = (float)(scale / s);
        }
    };
    const int nt = (int)std::max(1u, std::min(16u, std::thread::hardware_concurrency()));
    std::vector<std::thread> pool;
    const long long chunk = (M + nt - 1) / nt;
    for (int t = 0; t < nt; ++t)
        pool.emplace_back(work, std::min(M, t * chunk), std::min(M, (t + 1) * chunk));
    for (auto &th : pool) th.join();
}

void build_filter_basis(int n, int order, std::vector<float> &q)
{
    const int nq = std::min(order, FILTER_MAXQ - 1) + 1;
    std::vector<std::vector<double>> b(nq, std::vector<double>((size_t)n));
    for (int d = 0; d < nq; ++d) {
        for (int s = 0; s < n; ++s) {
            const double t = n > 1 ? -1.0 + 2.0 * (double)s / (double)(n - 1) : 0.0;
            b[d][s] = std::pow(t, d);
        }
        for (int pass = 0; pass < 2; ++pass)                     // modified Gram-Schmidt, twice
            for (int e = 0; e < d; ++e) {
                double dot = 0.0;
                for (int s = 0; s < n; ++s) dot += b[e][s] * b[d][s];
                for (int s = 0; s < n; ++s) b[d][s] -= dot * b[e][s];
            }
        double nrm = 0.0;
        for (int s = 0; s < n; ++s) nrm += b[d][s] * b[d][s];
        nrm = std::sqrt(nrm);
        // more basis functions than points: the remaining ones vanish (the fit is exact already)
        for (int s = 0; s < n; ++s) b[d][s] = (nrm > 1e-12 * std::sqrt((double)n)) ? b[d][s] / nrm : 0.0;
    }
    q.assign((size_t)n * FILTER_MAXQ, 0.f);
    for (int d = 0; d < nq; ++d)
        for (int s = 0; s < n; ++s) q[(size_t)s * FILTER_MAXQ + d] = (float)b[d][s];
}

void build_twiddles(int L, std::vector<float> &tw)
{
    tw.resize(2 * (size_t)L);
    for (int q = 0; q < L; ++q) {
        const double ang = 2.0 * kPi * (double)q / (double)L;
        tw[2 * q] = (float)std::cos(ang);
        tw[2 * q + 1] = (float)(-std::sin(ang));
    }
}

// iterative radix-2 FFT in double (plan time only; L is a power of two)
static void host_fft(std::vector<double> &re, std::vector<double> &im)
{
    const int L = (int)re.size();
    for (int i = 1, j = 0; i < L; ++i) {
        int bit = L >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { std::swap(re[i], re[j]); std::swap(im[i], im[j]); }
    }
    for (int len = 2; len <= L; len <<= 1) {
        for (int i = 0; i < L; i += len)
            for (int k = 0; k < len / 2; ++k) {
                const double ang = -2.0 * kPi * (double)k / (double)len;
                const double wr = std::cos(ang), wi = std::sin(ang);
                const int p = i + k, q = p + len / 2;
                const double tr = re[q] * wr - im[q] * wi, ti = re[q] * wi + im[q] * wr;
                re[q] = re[p] - tr; im[q] = im[p] - ti;
                re[p] += tr; im[p] += ti;
            }
    }
}

static inline long long posmod(long long v, long long m)
{
    long long r = v % m;
    return r < 0 ? r + m : r;
}

void build_chirp(int n, int L, std::vector<float> &a, std::vector<float> &b, std::vector<float> &hf)
{
    // Centred DFT  Z[k] = (1/n) sum_s z[s] exp(-i 2 pi (k-c)(s-c)/n),  c = n/2.
    //   (k-c)(s-c) = ks - c(k+s) + c^2
    // direct (L == n):     a[s] = exp(+i 2 pi c s/n),  b[k] = (1/n) exp(+i 2 pi (c k - c^2)/n)
    // Bluestein (L > n):   ks = (k^2 + s^2 - (k-s)^2)/2
    //   a[s] = exp(i pi (-s^2 + 2 c s)/n), b[k] = (1/n) exp(i pi (-k^2 + 2 c k - 2 c^2)/n),
    //   h[d] = exp(+i pi d^2/n), Z = b .* (a.*z (*) h); hf = FFT_L(h)/L.
    const long long c = n / 2, n2 = 2LL * n;
    const bool direct = (L == n);
    a.resize(2 * (size_t)n); b.resize(2 * (size_t)n);
    for (long long s = 0; s < n; ++s) {
        const long long pa = direct ? posmod(2 * c * s, n2) : posmod(-s * s + 2 * c * s, n2);
        const long long pb = direct ? posmod(2 * c * s - 2 * c * c, n2)
                                    : posmod(-s * s + 2 * c * s - 2 * c * c, n2);
        const double aa = kPi * (double)pa / (double)n, ab = kPi * (double)pb / (double)n;
        a[2 * s] = (float)std::cos(aa); a[2 * s + 1] = (float)std::sin(aa);
        b[2 * s] = (float)(std::cos(ab) / n); b[2 * s + 1] = (float)(std::sin(ab) / n);
    }
    hf.clear();
    if (direct) return;
    std::vector<double> hr(L, 0.0), hi(L, 0.0);
    for (long long d = -(n - 1); d <= n - 1; ++d) {
        const double ang = kPi * (double)posmod(d * d, n2) / (double)n;
        const int idx = (int)posmod(d, L);
        hr[idx] = std::cos(ang); hi[idx] = std::sin(ang);
    }
    host_fft(hr, hi);
    hf.resize(2 * (size_t)L);
    for (int q = 0; q < L; ++q) {
        hf[2 * q] = (float)(hr[q] / L);
        hf[2 * q + 1] = (float)(hi[q] / L);
    }
}

// ---------------------------------------------------------------- rounds ---------
struct Cand {
    uint32_t ak;
    int16_t lx, ly;
};

// Which base cells a new sample of the round may NOT take.  The scatter kernel accumulates a
// footprint one ROW at a time (W loads, W FMAs, W stores, then a warp barrier), so two lanes
// only collide if they touch the same cells within one row step: same base row and base
// columns closer than W.  (Footprints of a round may overlap otherwise: lane i's row step l
// and lane j's row step l' != l are separated by a barrier.)
struct Occupancy {          // one bitmap row per base row, up to 128 base columns
    uint64_t rows[SB_H_MAX > GT_ROWS_MAX ? SB_H_MAX : GT_ROWS_MAX][2];
    int kh = 5;                // W - 1
    void clear() { std::memset(rows, 0, sizeof(rows)); }
    bool overlaps(int lx, int ly) const
    {
        return (lx < 64 ? (rows[ly][0] >> lx) : (rows[ly][1] >> (lx - 64))) & 1u;
    }
    void mark(int lx, int ly)
    {
        const int lo = std::max(lx - kh, 0), hi = std::min(lx + kh, 127);
        unsigned __int128 m = ((((unsigned __int128)1) << (hi - lo + 1)) - 1) << lo;
        constexpr int NR = (int)(sizeof(rows) / sizeof(rows[0]));
        // a step covers SC_STEP_ROWS rows from each lane's own base row: base rows closer than
        // that share a row within a step
        for (int y = std::max(ly - (SC_STEP_ROWS - 1), 0); y <= std::min(ly + (SC_STEP_ROWS - 1), NR - 1); ++y) {
            rows[y][0] |= (uint64_t)m; rows[y][1] |= (uint64_t)(m >> 64);
        }
    }
};

// Greedy packing of `cands` (in order) into rounds of 32 lanes.  Appends 32 slots per
// round to `out`; returns the number of rounds.
static int build_rounds(std::vector<Cand> &cands, bool disjoint, int pitch, int W,
                        std::vector<Slot> &out, long long &filled)
{
    int rounds = 0;
    Occupancy occ;
    occ.kh = W - 1;
    std::vector<Cand> next;
    next.reserve(cands.size());
    while (!cands.empty()) {
        if (disjoint) occ.clear();
        uint32_t mask[2] = {0u, 0u};
        int cnt[2] = {0, 0};
        Slot lanes[32];
        for (int i = 0; i < 32; ++i) { lanes[i].ak = SLOT_EMPTY; lanes[i].lxy = 0; }
        next.clear();
        size_t i = 0;
        for (; i < cands.size(); ++i) {
            if (cnt[0] == 16 && cnt[1] == 16) break;
            const Cand &c = cands[i];
            const uint32_t res = 1u << ((c.ly * pitch + c.lx) & 15);
            int h = -1;
            if (cnt[0] < 16 && !(mask[0] & res)) h = 0;
            else if (cnt[1] < 16 && !(mask[1] & res)) h = 1;
            if (h < 0 || (disjoint && occ.overlaps(c.lx, c.ly))) { next.push_back(c); continue; }
            if (disjoint) occ.mark(c.lx, c.ly);
            mask[h] |= res;
            Slot &s = lanes[h * 16 + cnt[h]++];
            s.ak = c.ak;
            s.lxy = (uint32_t)c.lx | ((uint32_t)c.ly << 16);
        }
        for (; i < cands.size(); ++i) next.push_back(cands[i]);
        // Second pass: lanes still idle take candidates whose bank pair is already used ONCE in
        // their half-warp (a 2-way conflict costs that half-warp one extra wavefront per access;
        // an idle lane costs the whole round again later).  Footprint disjointness still holds.
        if (cnt[0] + cnt[1] < 32 && !next.empty()) {
            uint32_t twice[2] = {0u, 0u};
            size_t w = 0;
            for (size_t q = 0; q < next.size(); ++q) {
                const Cand &c = next[q];
                const uint32_t res = 1u << ((c.ly * pitch + c.lx) & 15);
                int h = -1;
                if (cnt[0] + cnt[1] < 32 && !(disjoint && occ.overlaps(c.lx, c.ly))) {
                    if (cnt[0] < 16 && !(twice[0] & res)) h = 0;
                    else if (cnt[1] < 16 && !(twice[1] & res)) h = 1;
                }
                if (h < 0) { next[w++] = c; continue; }
                if (disjoint) occ.mark(c.lx, c.ly);
                if (mask[h] & res) twice[h] |= res; else mask[h] |= res;
                Slot &sl = lanes[h * 16 + cnt[h]++];
                sl.ak = c.ak;
                sl.lxy = (uint32_t)c.lx | ((uint32_t)c.ly << 16);
            }
            next.resize(w);
        }
        filled += cnt[0] + cnt[1];
        out.insert(out.end(), lanes, lanes + 32);
        cands.swap(next);
        ++rounds;
    }
    return rounds;
}

static inline int floordiv(int a, int b) { return (a >= 0) ? a / b : -((-a + b - 1) / b); }

// ---------------------------------------------------------------- gather ---------
// Samples a schedule covers.  Full: every (a, k), k < n_det.  Hermitian half (real image /
// real sinogram: F[a,-j] = conj F[a,j]): the gather needs j >= 0 only, i.e. k in [n/2, n), plus,
// for even n, the GHOST k = n (j = +n/2), the mirror image of the unpaired j = -n/2.
static inline int half_k_begin(const Geometry &g) { return g.n_det / 2; }
static inline int half_k_end(const Geometry &g) { return g.n_det + ((g.n_det & 1) ? 0 : 1); }
// Samples the SCATTER schedules cover.  Full: k < n_det; Hermitian half: additionally the
// Nyquist ghost k = n_det (even n).  In both, j = 0 (k = n/2) is LEFT OUT: it sits at
// kappa = (0,0) for every angle, so its n_angles footprints coincide (they could only be
// accumulated one per round); dc_kernel sums the n_angles values first and adds one footprint.
static inline int scatter_k_end(const Geometry &g, bool half) { return half ? half_k_end(g) : g.n_det; }
static inline bool scatter_k_valid(const Geometry &g, int k) { return k != g.n_det / 2; }

// Items -> persistent CTAs of the gather (shared by the host and the device builder)
void finish_gather(Schedules &out, int n_workers)
{
    std::stable_sort(out.gather_ctas.begin(), out.gather_ctas.end(),
                     [](const GatherCta &x, const GatherCta &y) { return x.round_count > y.round_count; });
    // Items -> persistent CTAs: longest processing time first onto the least loaded worker
    // (deterministic: ties go to the lowest worker index), then grouped by worker.
    const int P = std::max(1, n_workers);
    std::vector<long long> load(P, 0);
    std::vector<std::vector<GatherCta>> mine(P);
    for (const GatherCta &c : out.gather_ctas) {
        int w = 0;
        for (int q = 1; q < P; ++q) if (load[q] < load[w]) w = q;
        load[w] += c.round_count + GATHER_ITEM_COST;
        mine[w].push_back(c);
    }
    out.gather_ctas.clear();
    out.gather_worker_begin.assign(1, 0);
    for (int w = 0; w < P; ++w) {
        // a worker's items arrive heaviest first; interleave them heavy, light, heavy, ... so
        // that the interpolation of a dense tile overlaps the staging of sparse ones (the
        // copy engine runs GATHER_STAGES items ahead)
        const std::vector<GatherCta> &m = mine[w];
        for (size_t lo = 0, hi = m.size(); lo < hi;) {
            out.gather_ctas.push_back(m[lo++]);
            if (lo < hi) out.gather_ctas.push_back(m[--hi]);
        }
        out.gather_worker_begin.push_back((int)out.gather_ctas.size());
    }
}


static void build_gather(const Geometry &g, Schedules &out, int n_workers)
{
    const int G = g.G, KW = g.W;
    const bool half = out.half;
    const int k0 = half ? half_k_begin(g) : 0, k1 = half ? half_k_end(g) : g.n_det, nk = k1 - k0;
    // half: bases of the j >= 0 samples lie in rows [G/2 - W/2, G - W/2]; tiles start there
    const int yorg = half ? (int)posmod(G / 2 - KW / 2, G) : 0;
    const int ntx = (G + GT_X - 1) / GT_X;
    const long long M = (long long)g.n_angles * nk;
    std::vector<uint32_t> tile_of(M);
    std::vector<Cand> all(M);
    int nty = 1;
    for (int a = 0; a < g.n_angles; ++a)
        for (int k = k0; k < k1; ++k) {
            int x0, y0;
            g.base(a, k, x0, y0);
            const int bx = (int)posmod(x0, G), by = (int)posmod(y0 - yorg, G);
            const int t = (by / GT_Y) * ntx + (bx / GT_X);
            nty = std::max(nty, by / GT_Y + 1);
            const long long m = (long long)a * nk + (k - k0);
            tile_of[m] = (uint32_t)t;
            all[m].ak = ((uint32_t)a << 16) | (uint32_t)k;
            all[m].lx = (int16_t)(bx % GT_X);
            all[m].ly = (int16_t)(by % GT_Y);
        }
    std::vector<uint32_t> count((size_t)ntx * nty + 1, 0);
    for (long long m = 0; m < M; ++m) ++count[tile_of[m] + 1];
    for (size_t t = 0; t < (size_t)ntx * nty; ++t) count[t + 1] += count[t];
    std::vector<uint32_t> order(M), fill(count.begin(), count.end() - 1);
    for (long long m = 0; m < M; ++m) order[fill[tile_of[m]]++] = (uint32_t)m;   // stable: (a,k) order

    std::vector<Cand> cands;
    for (int t = 0; t < ntx * nty; ++t) {
        if (count[t + 1] == count[t]) continue;
        cands.clear();
        for (uint32_t q = count[t]; q < count[t + 1]; ++q) cands.push_back(all[order[q]]);
        const int rb = (int)(out.gather_slots.size() / 32);
        const int nr = build_rounds(cands, false, gt_pitch(KW), KW, out.gather_slots, out.gather_filled);
        for (int r = 0; r < nr; r += GATHER_ROUND_CAP) {
            GatherCta c;
            c.tx0 = (t % ntx) * GT_X; c.ty0 = (int)posmod(yorg + (t / ntx) * GT_Y, G);
            c.round_begin = rb + r;
            c.round_count = std::min(GATHER_ROUND_CAP, nr - r);
            out.gather_ctas.push_back(c);
        }
    }
    finish_gather(out, n_workers);
}

// ---------------------------------------------------------------- scatter --------
struct Image { uint32_t ak; int bx, by; };   // one wrap image of a sample: base cell (may be < 0)

// Output rows a scatter schedule produces.  Full: [0, G).  Hermitian half (real sinogram: the
// gridded spectrum is Hermitian, the 2-D inverse FFT reads ky = 0 .. G/2 only): centred rows
// [G/2, G) and row 0 (ky = -G/2 == +G/2).  Samples: every (a, k), k < n_det, plus, for even n,
// the ghost k = n (the kernel gives it half the conjugated value of k = 0, and k = 0 half its
// own: Re{.} of the unpaired Nyquist sample).
struct RowSeg { int y0, y1; };
struct RectGeom { int rx0, ry0, rw, rh; };

static void scatter_rects(const Geometry &g, bool half, std::vector<RowSeg> &segs, std::vector<RectGeom> &rects,
                          std::vector<int> &seg_first)
{
    const int G = g.G;
    segs.clear(); rects.clear(); seg_first.clear();
    if (half) { segs.push_back(RowSeg{0, 1}); segs.push_back(RowSeg{G / 2, G}); }
    else segs.push_back(RowSeg{0, G});
    for (const RowSeg &sg : segs) {
        seg_first.push_back((int)rects.size());
        for (int ry0 = sg.y0; ry0 < sg.y1; ry0 += g.sr_y())
            for (int rx0 = 0; rx0 < G; rx0 += SR_X)
                rects.push_back(RectGeom{rx0, ry0, std::min(SR_X, G - rx0), std::min(g.sr_y(), sg.y1 - ry0)});
    }
}

static void build_scatter(const Geometry &g, Schedules &out, int n_workers)
{
    const int G = g.G, KW = g.W, KH = KW - 1;
    const bool half = out.half;
    const int k_end = scatter_k_end(g, half);
    int round_max = SCATTER_ROUND_MAX;       // set below, once the incidences are counted
    const int nrx = (G + SR_X - 1) / SR_X;
    std::vector<RowSeg> segs;
    std::vector<RectGeom> rects;
    std::vector<int> seg_first;
    scatter_rects(g, half, segs, rects, seg_first);
    const int nrect = (int)rects.size();
    // pass 1: count incidences (image, rect); pass 2: fill
    std::vector<uint32_t> count((size_t)nrect + 1, 0);
    std::vector<Image> inc;
    for (int pass = 0; pass < 2; ++pass) {
        std::vector<uint32_t> fill;
        if (pass == 1) {
            for (int r = 0; r < nrect; ++r) count[r + 1] += count[r];
            inc.resize(count[nrect]);
            fill.assign(count.begin(), count.end() - 1);
        }
        for (int a = 0; a < g.n_angles; ++a)
            for (int k = 0; k < k_end; ++k) {
                if (!scatter_k_valid(g, k)) continue;
                int x0, y0;
                g.base(a, k, x0, y0);
                for (int sy = -1; sy <= 1; ++sy) {
                    const int by = y0 + sy * G;
                    if (by + KH < 0 || by > G - 1) continue;
                    for (int sx = -1; sx <= 1; ++sx) {
                        const int bx = x0 + sx * G;
                        if (bx + KH < 0 || bx > G - 1) continue;
                        const int rx_lo = std::max(bx, 0) / SR_X, rx_hi = std::min(bx + KH, G - 1) / SR_X;
                        for (size_t sg = 0; sg < segs.size(); ++sg) {
                            const int ylo = std::max(by, segs[sg].y0), yhi = std::min(by + KH, segs[sg].y1 - 1);
                            if (ylo > yhi) continue;
                            const int ry_lo = (ylo - segs[sg].y0) / g.sr_y(), ry_hi = (yhi - segs[sg].y0) / g.sr_y();
                            for (int ry = ry_lo; ry <= ry_hi; ++ry)
                                for (int rx = rx_lo; rx <= rx_hi; ++rx) {
                                    const int r = seg_first[sg] + ry * nrx + rx;
                                    if (pass == 0) ++count[r + 1];
                                    else inc[fill[r]++] = Image{((uint32_t)a << 16) | (uint32_t)k, bx, by};
                                }
                        }
                    }
                }
            }
    }

    // Rounds a warp runs before a tile's samples are split over several CTAs.  A tile that runs
    // alone takes ~0.4 us per round whatever the rest of the device does, so the limit follows the
    // load: about 1.8 x the mean number of rounds per resident warp (measured at config 4: 48 rounds
    // is best for the Hermitian-half schedule, mean 26.5, and 96 for the full one, mean 53; at the
    // small configs, where a handful of centre tiles hold most samples, the lower limit:
    // bare gridding at config 1 39 -> 15 us, config 3 51 -> 20 us).
    {
        long long est_rounds = 0;
        for (int r = 0; r < nrect; ++r) est_rounds += (count[r + 1] - count[r] + 27) / 28;
        round_max = scatter_round_limit(g, out.half, est_rounds, n_workers);
    }
    struct Pending { ScatterCta cta; long long work; };
    std::vector<Pending> ctas;
    std::vector<Cand> quad[SCATTER_ITEMS];
    std::vector<Slot> tmp_slots;

    for (int r = 0; r < nrect; ++r) {
        const int rx0 = rects[r].rx0, ry0 = rects[r].ry0, rw = rects[r].rw, rh = rects[r].rh;
        const int nsx = (rw + ST_X - 1) / ST_X, nsy = (rh + g.st_y - 1) / g.st_y;
        const uint32_t lo = count[r], hi = count[r + 1];

        // quadrants of the rectangle and, for each, every sample image whose footprint
        // intersects it (a sample near a quadrant border is listed in both: each warp applies
        // only the taps inside its own quadrant)
        ScatterItem geom[SCATTER_ITEMS];
        std::memset(geom, 0, sizeof(geom));
        for (auto &v : quad) v.clear();
        for (int iy = 0; iy < nsy; ++iy)
            for (int ix = 0; ix < nsx; ++ix) {
                ScatterItem &I = geom[iy * SQ_X + ix];
                I.sx0 = ix * ST_X; I.sy0 = iy * g.st_y;
                I.sw = std::min(ST_X, rw - I.sx0); I.sh = std::min(g.st_y, rh - I.sy0);
                const int ax0 = rx0 + I.sx0, ay0 = ry0 + I.sy0;          // absolute origin
                for (uint32_t q = lo; q < hi; ++q) {
                    const Image &im = inc[q];
                    if (im.bx + KH < ax0 || im.bx >= ax0 + I.sw || im.by + KH < ay0 || im.by >= ay0 + I.sh) continue;
                    Cand c;
                    c.ak = im.ak;
                    c.lx = (int16_t)(im.bx - (ax0 - KH));
                    c.ly = (int16_t)(im.by - (ay0 - KH));
                    quad[iy * SQ_X + ix].push_back(c);
                }
            }

        // K CTAs share the rectangle: each quadrant's samples are dealt round-robin over them
        size_t biggest = 0;
        for (auto &v : quad) biggest = std::max(biggest, v.size());
        int K = std::max<int>(1, (int)((biggest + (size_t)24 * round_max - 1) / ((size_t)24 * round_max)));
        // Rounds of a warp: first the footprints wholly inside its quadrant (no clipping: the
        // kernel runs them without tap predicates), then the clipped ones.
        std::vector<Cand> part, part_clip;
        std::vector<int> rb, rc, rf;
        long long f = 0;
        for (int attempt = 0; attempt < 8; ++attempt) {
            tmp_slots.clear(); f = 0;
            rb.assign((size_t)K * SCATTER_ITEMS, 0); rc.assign((size_t)K * SCATTER_ITEMS, 0);
            rf.assign((size_t)K * SCATTER_ITEMS, 0);
            int mr = 0;
            for (int kk = 0; kk < K; ++kk)
                for (int it = 0; it < SCATTER_ITEMS; ++it) {
                    part.clear(); part_clip.clear();
                    for (size_t q = kk; q < quad[it].size(); q += K) {
                        const Cand &c = quad[it][q];
                        const bool inside = c.lx >= KH && c.lx <= geom[it].sw - 1 && c.ly >= KH && c.ly <= geom[it].sh - 1;
                        (inside ? part : part_clip).push_back(c);
                    }
                    rb[kk * SCATTER_ITEMS + it] = (int)(tmp_slots.size() / 32);
                    // one greedy packing over "inside first, clipped after": the leading rounds
                    // come out all-inside, one round mixes, the rest is clipped
                    part.insert(part.end(), part_clip.begin(), part_clip.end());
                    const int nr = build_rounds(part, true, ACC_PITCH, KW, tmp_slots, f);
                    rc[kk * SCATTER_ITEMS + it] = nr;
                    int nf = 0;
                    for (; nf < nr; ++nf) {
                        const Slot *lanes = &tmp_slots[((size_t)rb[kk * SCATTER_ITEMS + it] + nf) * 32];
                        bool all_in = true;
                        for (int l = 0; l < 32 && all_in; ++l) {
                            if (lanes[l].ak == SLOT_EMPTY) continue;
                            const int lx = (int)(lanes[l].lxy & 0xffff), ly = (int)(lanes[l].lxy >> 16);
                            all_in = lx >= KH && lx <= geom[it].sw - 1 && ly >= KH && ly <= geom[it].sh - 1;
                        }
                        if (!all_in) break;
                    }
                    rf[kk * SCATTER_ITEMS + it] = RADON_SC_FAST ? nf : 0;
                    mr = std::max(mr, rc[kk * SCATTER_ITEMS + it]);
                }
            if (mr <= round_max || attempt == 7) break;
            K = (int)std::ceil(K * (double)mr / round_max * 1.1) + (attempt > 2);
        }
        const int base = (int)(out.scatter_slots.size() / 32);
        out.scatter_slots.insert(out.scatter_slots.end(), tmp_slots.begin(), tmp_slots.end());
        out.scatter_filled += f;
        // cells of the centre window (the footprint of the summed j = 0 samples, DESIGN.md R-tie;
        // rows ky >= 0 only on the half grid) in this rectangle: then it is a merge job even when
        // one CTA grids it, because the merge is where that sum is added
        bool has_dc = false;
        for (int uy = (half ? 0 : -KW / 2); uy <= KW / 2; ++uy)
            for (int ux = -KW / 2; ux <= KW / 2; ++ux) {
                const int cx = G / 2 + ux, cy = G / 2 + uy;
                has_dc = has_dc || (cx >= rx0 && cx < rx0 + rw && cy >= ry0 && cy < ry0 + rh);
            }
        int first_slot = -1, job = -1;
        if (K > 1 || has_dc) {
            first_slot = out.n_partial_slots;
            out.n_partial_slots += K;
            job = (int)out.merge_jobs.size();
            MergeJob mj{rx0, ry0, rw, rh, first_slot, K, K + (has_dc ? 1 : 0), 0};
            out.merge_jobs.push_back(mj);
            if (has_dc) out.dc_jobs.push_back(job);
        }
        for (int kk = 0; kk < K; ++kk) {
            Pending p;
            std::memset(&p.cta, 0, sizeof(p.cta));
            p.cta.rx0 = rx0; p.cta.ry0 = ry0; p.cta.rw = rw; p.cta.rh = rh;
            p.cta.partial_slot = (job >= 0) ? first_slot + kk : -1;
            p.cta.job = job;
            p.work = 0;
            for (int it = 0; it < SCATTER_ITEMS; ++it) {
                p.cta.items[it] = geom[it];
                p.cta.items[it].round_begin = base + rb[kk * SCATTER_ITEMS + it];
                p.cta.items[it].round_count = rc[kk * SCATTER_ITEMS + it];
                p.cta.items[it].fast_count = rf[kk * SCATTER_ITEMS + it];
                p.work = std::max<long long>(p.work, rc[kk * SCATTER_ITEMS + it]);
            }
            ctas.push_back(p);
        }
    }
    std::stable_sort(ctas.begin(), ctas.end(),
                     [](const Pending &x, const Pending &y) { return x.work > y.work; });
    out.scatter_ctas.reserve(ctas.size());
    for (auto &p : ctas) out.scatter_ctas.push_back(p.cta);
}

// ---------------------------------------------------------------- paper's bins ----
void build_paper_bins(const Geometry &g, int n_bins_target, PaperBins &out)
{
    const int G = g.G, KH = g.W - 1;
    struct Node { int x0, y0, w, h; std::vector<PaperBinEntry> e; };
    auto cost = [](const Node &n) { return (long long)n.e.size() * n.w * n.h; };
    auto base_of = [&](const PaperBinEntry &en, int &bx, int &by) {
        int x0, y0;
        g.base((int)(en.ak >> 16), (int)(en.ak & 0xffff), x0, y0);
        bx = x0 + ((en.shift & 3) - 1) * G;
        by = y0 + (((en.shift >> 2) & 3) - 1) * G;
    };
    std::vector<Node> nodes(1);
    nodes[0] = Node{0, 0, G, G, {}};
    for (int a = 0; a < g.n_angles; ++a)
        for (int k = 0; k < g.n_det; ++k) {
            int x0, y0;
            g.base(a, k, x0, y0);
            for (int sy = -1; sy <= 1; ++sy) {
                const int by = y0 + sy * G;
                if (by + KH < 0 || by > G - 1) continue;
                for (int sx = -1; sx <= 1; ++sx) {
                    const int bx = x0 + sx * G;
                    if (bx + KH < 0 || bx > G - 1) continue;
                    nodes[0].e.push_back(PaperBinEntry{((uint32_t)a << 16) | (uint32_t)k, (sx + 1) | ((sy + 1) << 2)});
                }
            }
        }
    // "recursively divides the most computationally intensive bin into four equally sized bins"
    while ((int)nodes.size() < n_bins_target) {
        int top = -1;
        long long best = 0;
        for (size_t i = 0; i < nodes.size(); ++i)
            if (nodes[i].w >= 16 && nodes[i].h >= 16 && cost(nodes[i]) > best) { best = cost(nodes[i]); top = (int)i; }
        if (top < 0) break;
        Node parent = std::move(nodes[top]);
        nodes[top] = std::move(nodes.back());
        nodes.pop_back();
        const int hw = parent.w / 2, hh = parent.h / 2;
        for (int qy = 0; qy < 2; ++qy)
            for (int qx = 0; qx < 2; ++qx) {
                Node c{parent.x0 + qx * hw, parent.y0 + qy * hh, qx ? parent.w - hw : hw, qy ? parent.h - hh : hh, {}};
                for (const PaperBinEntry &en : parent.e) {
                    int bx, by;
                    base_of(en, bx, by);
                    if (bx + KH >= c.x0 && bx < c.x0 + c.w && by + KH >= c.y0 && by < c.y0 + c.h) c.e.push_back(en);
                }
                nodes.push_back(std::move(c));
            }
    }
    std::stable_sort(nodes.begin(), nodes.end(), [&](const Node &a, const Node &b) { return cost(a) > cost(b); });
    out.bins.clear(); out.entries.clear();
    for (const Node &n : nodes) {
        out.bins.push_back(PaperBin{n.x0, n.y0, n.w, n.h, (int)out.entries.size(), (int)n.e.size()});
        out.entries.insert(out.entries.end(), n.e.begin(), n.e.end());
    }
}

// ---- helpers shared with the device builder (plan_device.cu) -------------------------------------
void scatter_tile_rects(const Geometry &g, bool half, std::vector<TileRect> &tiles)
{
    std::vector<RowSeg> segs;
    std::vector<RectGeom> rects;
    std::vector<int> seg_first;
    scatter_rects(g, half, segs, rects, seg_first);
    tiles.clear();
    for (const RectGeom &r : rects) tiles.push_back(TileRect{r.rx0, r.ry0, r.rw, r.rh});
}

void sample_ranges(const Geometry &g, bool half, int &gather_k0, int &gather_k1, int &scatter_k1)
{
    gather_k0 = half ? half_k_begin(g) : 0;
    gather_k1 = half ? half_k_end(g) : g.n_det;
    scatter_k1 = scatter_k_end(g, half);
}

int scatter_round_limit(const Geometry &g, bool half, long long est_rounds, int n_workers)
{
    const double slots = (double)std::max(1, n_workers) * g.scatter_ctas_per_sm() * SCATTER_ITEMS;
    const int r = (int)std::lround(g.scatter_rfac(half) * (double)est_rounds / slots);
    return std::max(SCATTER_ROUND_MIN, std::min(SCATTER_ROUND_MAX, r));
}

void build_schedules(const Geometry &g, Schedules &out, bool half, int n_workers)
{
    out = Schedules();
    out.half = half;
    build_gather(g, out, n_workers);
    build_scatter(g, out, n_workers);
}

// ---------------------------------------------------------------- self check -----
static inline uint64_t tap_hash(uint32_t ak, int tx, int ty)
{
    uint64_t h = (uint64_t)ak * 0x9E3779B97F4A7C15ull + (uint64_t)(ty * KW_MAX + tx + 1) * 0xC2B2AE3D27D4EB4Full;
    h ^= h >> 29;
    return h | 1ull;
}

long long check_schedules(const Geometry &g, const Schedules &s)
{
    long long bad = 0;
    const int G = g.G, KW = g.W, KH = KW - 1;
    const bool half = s.half;
    const int kg0 = half ? half_k_begin(g) : 0, kg1 = half ? half_k_end(g) : g.n_det;   // gather samples
    const int ks1 = scatter_k_end(g, half);                                              // scatter samples
    const int nkg = kg1 - kg0;
    const long long M = (long long)g.n_angles * nkg;
    auto row_needed = [&](int cy) { return !half || cy == 0 || cy >= G / 2; };

    // Pairwise (brute force, independent of the builder's bitmap): at most two lanes of a
    // half-warp per bank pair; for the scatter, no two lanes of a round with the same base row and base
    // columns closer than W (the kernel's row-step rule), and every footprint inside the
    // accumulator.
    auto check_round = [&](const Slot *lanes, int pitch, bool disjoint) {
        for (int i = 0; i < 32; ++i) {
            if (lanes[i].ak == SLOT_EMPTY) continue;
            const int xi = lanes[i].lxy & 0xffff, yi = lanes[i].lxy >> 16;
            if (disjoint && (xi >= ST_X + KH || yi >= g.st_y + KH)) ++bad;
            int same_bank = 0;      // lanes of this half-warp in the same bank pair: at most 2-way
            for (int j = 0; j < 32; ++j)
                if (j != i && lanes[j].ak != SLOT_EMPTY && (i >> 4) == (j >> 4) &&
                    ((yi * pitch + xi) & 15) == ((int)((lanes[j].lxy >> 16) * pitch + (lanes[j].lxy & 0xffff)) & 15)) ++same_bank;
            if (same_bank > 1) ++bad;
            for (int j = i + 1; j < 32; ++j) {
                if (lanes[j].ak == SLOT_EMPTY) continue;
                const int xj = lanes[j].lxy & 0xffff, yj = lanes[j].lxy >> 16;
                if (disjoint && std::abs(yi - yj) < SC_STEP_ROWS && std::abs(xi - xj) < KW) ++bad;
            }
        }
    };

    // gather: the worker partition covers every item once, in order
    if (s.gather_worker_begin.empty() || s.gather_worker_begin.front() != 0 ||
        s.gather_worker_begin.back() != (int)s.gather_ctas.size()) ++bad;
    for (size_t w = 1; w < s.gather_worker_begin.size(); ++w)
        if (s.gather_worker_begin[w] < s.gather_worker_begin[w - 1]) ++bad;
    // gather: every sample exactly once, at the right place
    std::vector<uint8_t> seen(M, 0);
    for (const GatherCta &c : s.gather_ctas) {
        if (c.tx0 % GT_X || c.tx0 < 0 || c.ty0 < 0 || c.tx0 >= G || c.ty0 >= G) ++bad;
        if (c.round_count < 1 || c.round_count > GATHER_ROUND_CAP) ++bad;
        for (int r = 0; r < c.round_count; ++r) {
            const Slot *lanes = &s.gather_slots[(size_t)(c.round_begin + r) * 32];
            check_round(lanes, gt_pitch(KW), false);
            for (int l = 0; l < 32; ++l) {
                if (lanes[l].ak == SLOT_EMPTY) continue;
                const int a = lanes[l].ak >> 16, k = lanes[l].ak & 0xffff;
                if (a >= g.n_angles || k < kg0 || k >= kg1) { ++bad; continue; }
                int x0, y0;
                g.base(a, k, x0, y0);
                const int lx = lanes[l].lxy & 0xffff, ly = lanes[l].lxy >> 16;
                if (lx >= GT_X || ly >= GT_Y) ++bad;
                if (posmod(c.tx0 + lx - x0, G) != 0 || posmod(c.ty0 + ly - y0, G) != 0) ++bad;
                if (seen[(size_t)a * nkg + (k - kg0)]++) ++bad;
            }
        }
    }
    for (long long m = 0; m < M; ++m) if (!seen[m]) ++bad;

    // scatter: simulate with hashed unit weights and compare with the definition
    std::vector<uint64_t> expect((size_t)G * G, 0), got((size_t)G * G, 0);
    std::vector<uint8_t> written((size_t)G * G, 0);
    for (int a = 0; a < g.n_angles; ++a)
        for (int k = 0; k < ks1; ++k) {
            if (!scatter_k_valid(g, k)) continue;
            int x0, y0;
            g.base(a, k, x0, y0);
            const uint32_t ak = ((uint32_t)a << 16) | (uint32_t)k;
            for (int ty = 0; ty < KW; ++ty)
                for (int tx = 0; tx < KW; ++tx) {
                    const int cy = (int)posmod(y0 + ty, G);
                    if (row_needed(cy)) expect[(size_t)cy * G + posmod(x0 + tx, G)] += tap_hash(ak, tx, ty);
                }
        }
    std::vector<int> slot_owner(s.n_partial_slots, 0);
    for (const ScatterCta &c : s.scatter_ctas) {
        if (c.rx0 < 0 || c.ry0 < 0 || c.rx0 + c.rw > G || c.ry0 + c.rh > G || c.rw < 1 || c.rh < 1 ||
            c.rw > SR_X || c.rh > g.sr_y() || (c.rw & 1) || (c.rx0 & 1)) { ++bad; continue; }
        if (c.partial_slot >= 0) {
            if (c.partial_slot >= s.n_partial_slots) { ++bad; continue; }
            ++slot_owner[c.partial_slot];
        } else {
            for (int y = 0; y < c.rh; ++y)
                for (int x = 0; x < c.rw; ++x) ++written[(size_t)(c.ry0 + y) * G + c.rx0 + x];
        }
        // the warps' quadrants must be pairwise disjoint and inside the rectangle
        for (int i = 0; i < SCATTER_ITEMS; ++i) {
            const ScatterItem &A = c.items[i];
            if (A.round_count == 0) continue;
            if (A.sx0 < 0 || A.sy0 < 0 || A.sw < 1 || A.sh < 1 || A.sx0 + A.sw > c.rw || A.sy0 + A.sh > c.rh ||
                A.sw > ST_X || A.sh > g.st_y) ++bad;
            for (int j = i + 1; j < SCATTER_ITEMS; ++j) {
                const ScatterItem &B = c.items[j];
                if (B.round_count == 0) continue;
                if (A.sx0 < B.sx0 + B.sw && B.sx0 < A.sx0 + A.sw && A.sy0 < B.sy0 + B.sh && B.sy0 < A.sy0 + A.sh) ++bad;
            }
        }
        for (int it = 0; it < SCATTER_ITEMS; ++it) {
            const ScatterItem &I = c.items[it];
            if (I.round_count > SCATTER_ROUND_MAX * 2) ++bad;
            if (I.fast_count < 0 || I.fast_count > I.round_count) ++bad;
            const int ax0 = c.rx0 + I.sx0, ay0 = c.ry0 + I.sy0;
            for (int r = 0; r < I.round_count; ++r) {
                const Slot *lanes = &s.scatter_slots[(size_t)(I.round_begin + r) * 32];
                check_round(lanes, ACC_PITCH, true);
                for (int l = 0; l < 32; ++l) {
                    if (lanes[l].ak == SLOT_EMPTY) continue;
                    const int a = lanes[l].ak >> 16, k = lanes[l].ak & 0xffff;
                    if (a >= g.n_angles || k >= ks1 || !scatter_k_valid(g, k)) { ++bad; continue; }
                    int x0, y0;
                    g.base(a, k, x0, y0);
                    const int bx = ax0 - KH + (int)(lanes[l].lxy & 0xffff), by = ay0 - KH + (int)(lanes[l].lxy >> 16);
                    if (posmod(bx - x0, G) != 0 || posmod(by - y0, G) != 0) ++bad;
                    // fast rounds run without tap predicates: the footprint must lie inside the quadrant
                    if (r < I.fast_count && (bx < ax0 || bx + KH >= ax0 + I.sw || by < ay0 || by + KH >= ay0 + I.sh)) ++bad;
                    for (int ty = 0; ty < KW; ++ty)
                        for (int tx = 0; tx < KW; ++tx) {
                            const int cx = bx + tx, cy = by + ty;       // the kernel clips to the quadrant
                            if (cx < ax0 || cx >= ax0 + I.sw || cy < ay0 || cy >= ay0 + I.sh) continue;
                            got[(size_t)cy * G + cx] += tap_hash(lanes[l].ak, tx, ty);
                        }
                }
            }
        }
    }
    {   // every cell of the centre window lies in exactly one dc job; tickets are consistent
        if ((int)s.dc_jobs.size() > MAX_DC_JOBS) ++bad;
        std::vector<int> is_dc(s.merge_jobs.size(), 0);
        for (int j : s.dc_jobs) { if (j < 0 || j >= (int)s.merge_jobs.size()) { ++bad; continue; } ++is_dc[j]; }
        for (size_t j = 0; j < s.merge_jobs.size(); ++j)
            if (is_dc[j] > 1 || s.merge_jobs[j].expected != s.merge_jobs[j].n_slots + is_dc[j]) ++bad;
        for (int uy = (half ? 0 : -KW / 2); uy <= KW / 2; ++uy)
            for (int ux = -KW / 2; ux <= KW / 2; ++ux) {
                const int cx = G / 2 + ux, cy = G / 2 + uy;
                int n = 0;
                for (int j : s.dc_jobs) {
                    if (j < 0 || j >= (int)s.merge_jobs.size()) continue;
                    const MergeJob &mj = s.merge_jobs[j];
                    n += (cx >= mj.rx0 && cx < mj.rx0 + mj.rw && cy >= mj.ry0 && cy < mj.ry0 + mj.rh) ? 1 : 0;
                }
                if (n != 1) ++bad;
            }
        for (const ScatterCta &c : s.scatter_ctas) {
            if ((c.partial_slot >= 0) != (c.job >= 0)) { ++bad; continue; }
            if (c.job < 0) continue;
            if (c.job >= (int)s.merge_jobs.size()) { ++bad; continue; }
            const MergeJob &mj = s.merge_jobs[c.job];
            if (c.partial_slot < mj.first_slot || c.partial_slot >= mj.first_slot + mj.n_slots ||
                c.rx0 != mj.rx0 || c.ry0 != mj.ry0 || c.rw != mj.rw || c.rh != mj.rh) ++bad;
        }
    }
    for (const MergeJob &mj : s.merge_jobs) {
        for (int i = 0; i < mj.n_slots; ++i)
            if (mj.first_slot + i >= s.n_partial_slots || slot_owner[mj.first_slot + i] != 1) ++bad;
        for (int y = 0; y < mj.rh; ++y)
            for (int x = 0; x < mj.rw; ++x) ++written[(size_t)(mj.ry0 + y) * G + mj.rx0 + x];
    }
    for (size_t i = 0; i < (size_t)G * G; ++i) {
        if (written[i] != (row_needed((int)(i / (size_t)G)) ? 1 : 0)) ++bad;
        if (got[i] != expect[i]) ++bad;
    }
    return bad;
}

}  // namespace radon
