// api.cu -- the C ABI of libradon_b200 (include/radon.h): plan life cycle and the stage
// sequences of radon_forward / radon_adjoint.  No torch types, no exceptions across the ABI.
#include "../../include/radon.h"

#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>

#include "kernels.h"
#include "plan_device.h"

using namespace radon;

static thread_local std::string g_last_cuda_error;

#define CUDA_TRY(expr)                                                                 \
    do {                                                                               \
        cudaError_t e__ = (expr);                                                      \
        if (e__ != cudaSuccess) {                                                      \
            g_last_cuda_error = std::string(#expr) + ": " + cudaGetErrorString(e__);   \
            return RADON_ECUDA;                                                        \
        }                                                                              \
    } while (0)

struct Workspace {
    float2 *T = nullptr;       // (G/2+1) x N Hermitian-half intermediate of the 2-D FFT
    float2 *grid = nullptr;    // G x G oversampled spectrum (centred)
    float2 *polar = nullptr;   // M polar samples
    float2 *dcbuf = nullptr;   // (W+1)^2 values: the summed j = 0 samples on the centre window
    float2 *scratch = nullptr; // partial rectangles of the scatter's split tiles (per workspace:
                               // two slices may be gridded at the same time on different streams)
    int *tickets = nullptr;    // counters of the merge jobs (zero between launches)
    float *img = nullptr;      // N x N   (host-buffer entry points only)
    float *sino = nullptr;     // M       (host-buffer entry points only)
};
constexpr int NWS = 4;         // workspaces = slices in flight of the host-buffer entry points

// Optional stage timing: one CUDA event at every stage boundary of forward / adjoint.
struct StageTimer {
    bool enabled = false;
    std::vector<cudaEvent_t> ev;      // pool, created on first enable
    std::vector<int> stage;           // stage id that STARTS at ev[i]; -1 = end of a sequence
    size_t used = 0;
    bool overflow = false;            // an event could not be created: the sample is truncated
    double acc_ms[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    long long cnt[8] = {0, 0, 0, 0, 0, 0, 0, 0};
};
constexpr size_t STAGE_EVENT_POOL = 8192;

struct radon_plan {
    StageTimer timer;
    Geometry geo;
    DevicePlan dev;
    Workspace ws[NWS];
    long long M = 0;
    int n_partial = 0;         // scratch slots a workspace needs (max over the two schedule sets)
    int n_jobs = 0;            // ticket counters a workspace needs (likewise)
    size_t device_bytes = 0;
    long long gather_slots[2] = {0, 0}, gather_filled[2] = {0, 0}, scatter_slots[2] = {0, 0}, scatter_filled[2] = {0, 0};
    cudaStream_t hstream[NWS] = {};
    cudaEvent_t hevent[NWS] = {};
    cudaEvent_t fork_event = nullptr;
    float *dev_density = nullptr;   // D of PAPER.md:89 times the quadrature scale, pair-symmetrised (density_setup)
    std::vector<float> host_density;   // the same table exactly as eq. :89 gives it (radon_plan_density)
    double density_scale = 0.0;
    // polynomial sinogram filter: orthonormal bases along the detector (n_det)
    // and along the angles (n_angles), built on first use or by radon_plan_set_filter
    int filter_order = -1;
    float *filter_q[2] = {nullptr, nullptr};
    // solver iteration: residual sinogram, and the iteration captured as a CUDA graph
    float *resid = nullptr;
    struct SolverGraph {
        cudaGraphExec_t exec = nullptr;
        const float *x = nullptr, *b = nullptr;
        float alpha = 0.f, tau = 0.f;
        int filtered = 0;
        long long kernels = 0;            // kernel nodes of one iteration
    } sgraph;
    cudaStream_t capture_stream = nullptr;
    // the paper's load-balanced bins (comparison variant, built on first use)
    PaperBin *pb_bins = nullptr;
    PaperBinEntry *pb_entries = nullptr;
    int pb_n_bins = 0, pb_target = 0, pb_max_samples = 0, pb_unstaged = 0;
    long long pb_n_entries = 0;
    // P3: where the schedules were built (1: CUDA kernels of plan_device.cu, 0: host builder) and the
    // host copy of everything but the slot arrays (radon_plan_schedule_check downloads those)
    int device_built[2] = {0, 0};
    Schedules meta[2];
    double schedule_ms = 0.0;
};

template <typename T>
static int dev_alloc(radon_plan *p, T **ptr, size_t count)
{
    *ptr = nullptr;
    if (count == 0) return RADON_OK;
    cudaError_t e = cudaMalloc((void **)ptr, count * sizeof(T));
    if (e != cudaSuccess) {
        g_last_cuda_error = std::string("cudaMalloc: ") + cudaGetErrorString(e);
        return e == cudaErrorMemoryAllocation ? RADON_ENOMEM : RADON_ECUDA;
    }
    p->device_bytes += count * sizeof(T);
    return RADON_OK;
}

template <typename T, typename H>
static int dev_upload(radon_plan *p, T **ptr, const std::vector<H> &host)
{
    static_assert(sizeof(T) % sizeof(H) == 0 || sizeof(H) % sizeof(T) == 0, "layout");
    const size_t bytes = host.size() * sizeof(H);
    int rc = dev_alloc(p, (unsigned char **)ptr, bytes);
    if (rc) return rc;
    if (bytes) CUDA_TRY(cudaMemcpy(*ptr, host.data(), bytes, cudaMemcpyHostToDevice));
    return RADON_OK;
}

static int validate(int N, int n_angles, int n_det, float sigma, int W, int *G_out)
{
    if (N < 8 || n_angles < 1 || n_det < 2 || n_angles > 65535 || n_det > 65533) return RADON_EINVAL;
    if (W < 2 || W > 12) return RADON_EINVAL;
    if (!(sigma > 1.0f) || sigma > 8.0f) return RADON_EINVAL;
    const double g = (double)sigma * N;
    const long long G = llround(g);
    if (fabs(g - (double)G) > 1e-6 || (G & 1)) return RADON_EINVAL;
    if (!kw_supported(W)) return RADON_EUNSUPPORTED;
    if (!fft_length_supported((int)G)) return RADON_EUNSUPPORTED;
    {   // projection DFT: one FFT of length n_det when that is a power of two >= 16, else Bluestein (L >= 2n - 1)
        const bool pow2 = (n_det & (n_det - 1)) == 0 && n_det >= 16;
        if (pow2 ? n_det > 8192 : 2 * (long long)n_det - 1 > 8192) return RADON_EUNSUPPORTED;
    }
    *G_out = (int)G;
    return RADON_OK;
}

extern "C" int radon_plan_destroy(radon_plan *p)
{
    if (!p) return RADON_OK;
    cudaDeviceSynchronize();
    DevicePlan &d = p->dev;
    cudaFree(d.cs); cudaFree(d.deapod); cudaFree(d.tw_G); cudaFree(d.tw_sub); cudaFree(d.tw_P);
    cudaFree(d.chirp_a); cudaFree(d.chirp_b); cudaFree(d.chirp_hf);
    for (auto &q : d.sched) {
        cudaFree(q.gather_ctas); cudaFree(q.gather_worker_begin); cudaFree(q.gather_slots); cudaFree(q.scatter_ctas); cudaFree(q.scatter_slots);
        cudaFree(q.merge_jobs);
    }
    for (auto &w : p->ws) { cudaFree(w.T); cudaFree(w.grid); cudaFree(w.polar); cudaFree(w.scratch); cudaFree(w.tickets); cudaFree(w.dcbuf); cudaFree(w.img); cudaFree(w.sino); }
    for (cudaEvent_t e : p->timer.ev) cudaEventDestroy(e);
    if (p->fork_event) cudaEventDestroy(p->fork_event);
    cudaFree(p->dev_density);
    cudaFree(p->filter_q[0]); cudaFree(p->filter_q[1]); cudaFree(p->resid);
    cudaFree(p->pb_bins); cudaFree(p->pb_entries);
    if (p->sgraph.exec) cudaGraphExecDestroy(p->sgraph.exec);
    if (p->capture_stream) cudaStreamDestroy(p->capture_stream);
    for (int i = 0; i < NWS; ++i) {
        if (p->hstream[i]) cudaStreamDestroy(p->hstream[i]);
        if (p->hevent[i]) cudaEventDestroy(p->hevent[i]);
    }
    delete p;
    return RADON_OK;
}

static int workspace_alloc(radon_plan *p, Workspace &w)
{
    const int G = p->dev.G, N = p->dev.N;
    int rc;
    if (!w.T && (rc = dev_alloc(p, &w.T, (size_t)(G / 2 + 1) * N))) return rc;
    if (!w.grid && (rc = dev_alloc(p, &w.grid, (size_t)G * G))) return rc;
    if (!w.polar && (rc = dev_alloc(p, &w.polar, (size_t)p->M))) return rc;
    if (!w.scratch && (rc = dev_alloc(p, &w.scratch, (size_t)std::max(p->n_partial, 1) * SR_X * p->geo.sr_y()))) return rc;
    if (!w.dcbuf && (rc = dev_alloc(p, &w.dcbuf, (size_t)(KW_MAX + 1) * (KW_MAX + 1)))) return rc;
    if (!w.tickets) {
        const size_t n = (size_t)std::max(p->n_jobs, 1) * MERGE_COUNTERS_PER_JOB;
        if ((rc = dev_alloc(p, &w.tickets, n))) return rc;
        CUDA_TRY(cudaMemset(w.tickets, 0, n * sizeof(int)));
    }
    return RADON_OK;
}

static int plan_create_impl(radon_plan *p, int N, int n_angles, int n_det, float sigma, int W, int G)
{
    int devid = 0;
    CUDA_TRY(cudaGetDevice(&devid));
    cudaDeviceProp prop;
    CUDA_TRY(cudaGetDeviceProperties(&prop, devid));
    if (prop.major != 10) return RADON_EARCH;          // sm_100a only: no other backend
    if (init_kernel_attributes()) { g_last_cuda_error = "cudaFuncSetAttribute(max dynamic smem)"; return RADON_ECUDA; }

    p->geo.init(N, n_angles, n_det, (double)sigma, W);
    p->M = (long long)n_angles * n_det;
    DevicePlan &d = p->dev;
    d.N = N; d.G = G; d.n_angles = n_angles; d.n_det = n_det; d.W = W; d.st_y = p->geo.st_y;
    d.n_sm = prop.multiProcessorCount;
    d.pdl = true;   // every kernel of a call waits (griddepcontrol.wait) for its predecessor and signals its dependents late
    const bool pow2 = (n_det & (n_det - 1)) == 0 && n_det >= 16;
    d.LP = pow2 ? n_det : std::max(16, next_pow2(2 * n_det - 1));

    int rc;
    // P1: Fourier-slice directions, fp64
    if ((rc = dev_upload(p, &d.cs, p->geo.cs))) return rc;
    // P2: Kaiser-Bessel polynomial pieces, de-apodisation
    std::vector<float> deapod, tw, ca, cb, hf;
    build_kb_poly(W, sigma, d.kb);
    build_deapod(N, G, W, sigma, deapod);
    if ((rc = dev_upload(p, &d.deapod, deapod))) return rc;
    build_twiddles(G, tw);
    if ((rc = dev_upload(p, &d.tw_G, tw))) return rc;
    {
        int P = 0, PR = 0;
        if ((G & (G - 1)) != 0 && fft_composite_split(G, &P, &PR)) {
            build_twiddles(P, tw);
            if ((rc = dev_upload(p, &d.tw_sub, tw))) return rc;
        }
    }
    build_twiddles(d.LP, tw);
    if ((rc = dev_upload(p, &d.tw_P, tw))) return rc;
    build_chirp(n_det, d.LP, ca, cb, hf);
    if ((rc = dev_upload(p, &d.chirp_a, ca))) return rc;
    if ((rc = dev_upload(p, &d.chirp_b, cb))) return rc;
    if (!hf.empty() && (rc = dev_upload(p, &d.chirp_hf, hf))) return rc;
    // P3: schedules
    int n_partial = 0;
    const char *builder_env = std::getenv("RADON_PLAN_BUILDER");          // "host": force the host builder
    const bool want_device = !(builder_env && std::strcmp(builder_env, "host") == 0);
    const auto t_sched = std::chrono::steady_clock::now();
    for (int h = 0; h < 2; ++h) {
        Schedules &sch = p->meta[h];
        DevicePlan::Sched &q = d.sched[h];
        Slot *dg = nullptr, *dsl = nullptr;
        long long ng = 0, ns = 0;
        int drc = want_device ? build_schedules_device(p->geo, d.cs, h == 1, d.n_sm, sch, &dg, &ng, &dsl, &ns) : -3;
        if (drc == 0) {
            p->device_built[h] = 1;
            q.gather_slots = dg; q.scatter_slots = dsl;
            p->device_bytes += (size_t)(ng + ns) * 32 * sizeof(Slot);
            p->gather_slots[h] = ng * 32; p->scatter_slots[h] = ns * 32;
        } else {
            cudaGetLastError();                                          // a failed device build must not poison later calls
            build_schedules(p->geo, sch, h == 1, d.n_sm);
            p->gather_slots[h] = (long long)sch.gather_slots.size();
            p->scatter_slots[h] = (long long)sch.scatter_slots.size();
            if ((rc = dev_upload(p, &q.gather_slots, sch.gather_slots))) return rc;
            if ((rc = dev_upload(p, &q.scatter_slots, sch.scatter_slots))) return rc;
            sch.gather_slots.clear(); sch.gather_slots.shrink_to_fit();
            sch.scatter_slots.clear(); sch.scatter_slots.shrink_to_fit();
        }
        p->gather_filled[h] = sch.gather_filled;
        p->scatter_filled[h] = sch.scatter_filled;
        q.n_gather_ctas = (int)sch.gather_ctas.size();
        q.n_scatter_ctas = (int)sch.scatter_ctas.size();
        q.n_merge_jobs = (int)sch.merge_jobs.size();
        q.n_dc_jobs = (int)sch.dc_jobs.size();
        if (q.n_dc_jobs > MAX_DC_JOBS) return RADON_EINVAL;
        for (int i = 0; i < q.n_dc_jobs; ++i) q.dc_jobs[i] = sch.dc_jobs[i];
        if ((rc = dev_upload(p, &q.gather_ctas, sch.gather_ctas))) return rc;
        q.n_gather_workers = (int)sch.gather_worker_begin.size() - 1;
        if ((rc = dev_upload(p, &q.gather_worker_begin, sch.gather_worker_begin))) return rc;
        if ((rc = dev_upload(p, &q.scatter_ctas, sch.scatter_ctas))) return rc;
        if ((rc = dev_upload(p, &q.merge_jobs, sch.merge_jobs))) return rc;
        n_partial = std::max(n_partial, sch.n_partial_slots);
        p->n_jobs = std::max(p->n_jobs, (int)sch.merge_jobs.size());
    }
    p->schedule_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_sched).count();
    // workspaces: the first serves the device-pointer calls, all of them the host-buffer entry
    // points (copies and kernels of NWS slices overlap); allocated on first use beyond the first
    p->n_partial = n_partial;
    return workspace_alloc(p, p->ws[0]);
    return RADON_OK;
}

extern "C" int radon_plan_create(radon_plan **out, int N, int n_angles, int n_det, float sigma, int W)
{
    if (!out) return RADON_EINVAL;
    *out = nullptr;
    int G = 0;
    int rc = validate(N, n_angles, n_det, sigma, W, &G);
    if (rc) return rc;
    radon_plan *p = new (std::nothrow) radon_plan();
    if (!p) return RADON_ENOMEM;
    try {
        rc = plan_create_impl(p, N, n_angles, n_det, sigma, W, G);
    } catch (const std::bad_alloc &) {
        rc = RADON_ENOMEM;
    } catch (...) {
        rc = RADON_EINVAL;
    }
    if (rc) { radon_plan_destroy(p); return rc; }
    *out = p;
    return RADON_OK;
}

static int check_launch()
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        g_last_cuda_error = std::string("kernel launch: ") + cudaGetErrorString(e);
        return RADON_ECUDA;
    }
    return RADON_OK;
}

// ---- stage sequences ------------------------------------------------------------------
// stage ids: 0 F1 colpass_fwd, 1 F2 rowpass_fwd, 2 F3 gather, 3 F4 proj_ifft,
//            4 A1 proj_fft, 5 A2 scatter(+merge), 6 A3 rowpass_inv, 7 A4 colpass_inv
static inline void mark(radon_plan *p, cudaStream_t st, int stage)
{
    StageTimer &t = p->timer;
    if (!t.enabled) return;
    if (t.used >= t.ev.size()) {                 // pool full: grow it (measurement mode only)
        const size_t n = t.ev.size() + STAGE_EVENT_POOL;
        t.ev.resize(n, nullptr);
        t.stage.resize(n, -1);
        for (size_t i = t.used; i < n; ++i)
            if (cudaEventCreate(&t.ev[i]) != cudaSuccess) { t.ev.resize(i); t.stage.resize(i); break; }
        if (t.used >= t.ev.size()) { t.overflow = true; return; }
    }
    cudaEventRecord(t.ev[t.used], st);
    t.stage[t.used++] = stage;
}

// half: Hermitian-half schedules (d_polar then holds k >= n/2 of every row, and k = 0 for even n)
static int nufft2_ws(radon_plan *p, Workspace &w, bool half, const float *d_x, float2 *d_polar, cudaStream_t st)
{
    mark(p, st, 0);
    if (launch_fft2d_pass(0, p->dev, d_x, w.T, 0, st)) return RADON_ECUDA;                 // F1 + F2 (columns)
    mark(p, st, 1);
    if (launch_fft2d_pass(1, p->dev, w.T, w.grid, half ? 2 : 1, st)) return RADON_ECUDA;   // F2 (rows)
    mark(p, st, 2);
    if (launch_gather(p->dev, half, w.grid, d_polar, st)) return RADON_ECUDA;              // F3
    return check_launch();
}

// half: d_polar is Hermitian along every row (the DFT of a real sinogram); only the grid rows
// ky = 0 .. G/2 are gridded and the row pass reads them without folding.
static int nufft1_ws(radon_plan *p, Workspace &w, bool half, const float2 *d_polar, float *d_x, cudaStream_t st,
                     const IstaUpdate *upd = nullptr)
{
    mark(p, st, 5);
    if (launch_scatter(p->dev, half, d_polar, w.grid, w.scratch, w.dcbuf, w.tickets, st)) return RADON_ECUDA;             // A2
    mark(p, st, 6);
    if (launch_fft2d_pass(2, p->dev, w.grid, w.T, half ? 0 : 1, st)) return RADON_ECUDA;   // A3 (rows)
    mark(p, st, 7);
    if (launch_fft2d_pass(3, p->dev, w.T, d_x, 0, st, upd)) return RADON_ECUDA;   // A3 (columns) + A4 (+ solver update)
    return check_launch();
}

// ex.sub: the data, subtracted from the sinogram (residual); ex.q: filter basis (filter along the projections)
static int forward_ws(radon_plan *p, Workspace &w, const float *d_x, float *d_sino, cudaStream_t st,
                      const ProjExtra &ex = ProjExtra())
{
    int rc = nufft2_ws(p, w, true, d_x, w.polar, st);
    if (rc) return rc;
    mark(p, st, 3);
    if (launch_proj(true, true, p->dev, (const float *)w.polar, d_sino, nullptr, st, ex)) return RADON_ECUDA;   // F4
    mark(p, st, -1);
    return check_launch();
}

// dens == nullptr: the exact transpose of forward_ws (D == 1, reading S11); else the inverse
// Radon transform of PAPER.md:51 / :85 with the density compensation D of :89
static int adjoint_ws(radon_plan *p, Workspace &w, const float *d_sino, float *d_x, cudaStream_t st,
                      const float *dens = nullptr, const float *filter_q = nullptr, const IstaUpdate *upd = nullptr)
{
    mark(p, st, 4);
    ProjExtra ex;
    ex.q = filter_q;
    if (launch_proj(false, false, p->dev, d_sino, (float *)w.polar, dens, st, ex)) return RADON_ECUDA;  // A1
    int rc = check_launch();
    if (rc) return rc;
    rc = nufft1_ws(p, w, true, w.polar, d_x, st, upd);
    mark(p, st, -1);
    return rc;
}

extern "C" int radon_plan_stage_timing(radon_plan *p, int enable)
{
    if (!p) return RADON_EINVAL;
    StageTimer &t = p->timer;
    if (enable && t.ev.empty()) {
        t.ev.resize(STAGE_EVENT_POOL);
        t.stage.assign(STAGE_EVENT_POOL, -1);
        for (auto &e : t.ev) CUDA_TRY(cudaEventCreate(&e));
    }
    t.enabled = enable != 0;
    return RADON_OK;
}

extern "C" int radon_plan_stage_times(radon_plan *p, double total_ms[8], long long launches[8])
{
    if (!p) return RADON_EINVAL;
    StageTimer &t = p->timer;
    if (t.used) CUDA_TRY(cudaEventSynchronize(t.ev[t.used - 1]));
    for (size_t i = 0; i + 1 < t.used; ++i) {
        if (t.stage[i] < 0) continue;
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, t.ev[i], t.ev[i + 1]) == cudaSuccess) {
            t.acc_ms[t.stage[i]] += ms;
            t.cnt[t.stage[i]] += 1;
        }
    }
    t.used = 0;
    for (int s = 0; s < 8; ++s) {
        if (total_ms) total_ms[s] = t.acc_ms[s];
        if (launches) launches[s] = t.cnt[s];
        t.acc_ms[s] = 0; t.cnt[s] = 0;
    }
    const bool truncated = t.overflow;
    t.overflow = false;
    return truncated ? RADON_ENOMEM : RADON_OK;
}

extern "C" int radon_forward(radon_plan *p, const float *d_x, float *d_sino, void *stream)
{
    if (!p || !d_x || !d_sino) return RADON_EINVAL;
    return forward_ws(p, p->ws[0], d_x, d_sino, (cudaStream_t)stream);
}

extern "C" int radon_adjoint(radon_plan *p, const float *d_sino, float *d_x, void *stream)
{
    if (!p || !d_x || !d_sino) return RADON_EINVAL;
    return adjoint_ws(p, p->ws[0], d_sino, d_x, (cudaStream_t)stream);
}

// ---- inverse Radon transform ---------------------------------------
static int density_setup(radon_plan *p)
{
    if (p->dev_density) return RADON_OK;
    // D of eq. :89 on the device (plan_device.cu: one thread per sample, neighbours from the geometry,
    // fp64), downloaded once for radon_plan_density; RADON_PLAN_BUILDER=host builds it on the host.
    const int n = p->dev.n_det, na = p->dev.n_angles, W = p->geo.W;
    const double beta = kb_beta(W, p->geo.sigma), inv = 1.0 / kb_i0(beta);
    const double ph0 = (double)W * inv * std::sinh(beta) / beta;           // phihat(0): the integral of the kernel
    const double scale = (double)n * ph0 * ph0 / ((double)p->dev.G * (double)p->dev.G);
    const char *builder_env = std::getenv("RADON_PLAN_BUILDER");
    int rc;
    try {
        if (builder_env && std::strcmp(builder_env, "host") == 0) {
            build_density(p->geo, p->host_density, &p->density_scale);
            if ((rc = dev_upload(p, &p->dev_density, p->host_density))) return rc;
        } else {
            if ((rc = dev_alloc(p, &p->dev_density, (size_t)p->M))) return rc;
            if (launch_density(p->dev.cs, na, n, W, beta, inv, scale, p->dev_density, 0)) return RADON_ECUDA;
            p->host_density.resize((size_t)p->M);
            CUDA_TRY(cudaMemcpy(p->host_density.data(), p->dev_density, (size_t)p->M * sizeof(float), cudaMemcpyDeviceToHost));
            p->density_scale = scale;
        }
    } catch (const std::bad_alloc &) {
        return RADON_ENOMEM;
    }
    // radon_inverse runs the Hermitian-half scatter, which grids the pair (j, -j) as ONE complex
    // value and its conjugate: that is Re{D_j Yh_j e + D_-j conj(Yh_j) conj(e)} only if both
    // carry the same weight.  For odd n_det the sample set is point symmetric and D_j == D_-j;
    // for even n_det j = -n/2 has no partner and D_j != D_-j near the band edge.  The real part
    // only ever sees the pair sum (D_j + D_-j) Re{Yh_j e}, so giving both the mean is exact.
    if (launch_density_pair_mean(p->dev_density, na, n, 0)) return RADON_ECUDA;
    CUDA_TRY(cudaDeviceSynchronize());
    return RADON_OK;
}

// The blocking part of radon_inverse (the density table) done ahead of time, so that radon_inverse
// is asynchronous -- and capturable in a CUDA graph -- from its first call.
extern "C" int radon_plan_prepare_inverse(radon_plan *p)
{
    if (!p) return RADON_EINVAL;
    return density_setup(p);
}

extern "C" int radon_inverse(radon_plan *p, const float *d_sino, float *d_x, void *stream)
{
    if (!p || !d_x || !d_sino) return RADON_EINVAL;
    int rc = density_setup(p);
    if (rc) return rc;
    return adjoint_ws(p, p->ws[0], d_sino, d_x, (cudaStream_t)stream, p->dev_density);
}

extern "C" int radon_plan_density(radon_plan *p, float *h_density, double *scale)
{
    if (!p) return RADON_EINVAL;
    int rc = density_setup(p);
    if (rc) return rc;
    if (scale) *scale = p->density_scale;
    if (h_density) std::memcpy(h_density, p->host_density.data(), (size_t)p->M * sizeof(float));
    return RADON_OK;
}

extern "C" int radon_density_host(int N, int n_angles, int n_det, float sigma, int W, float *h_density, double *scale)
{
    if (!h_density) return RADON_EINVAL;
    int G = 0;
    int rc = validate(N, n_angles, n_det, sigma, W, &G);
    if (rc) return rc;
    try {
        Geometry geo;
        geo.init(N, n_angles, n_det, (double)sigma, W);
        std::vector<float> D;
        build_density(geo, D, scale);
        std::memcpy(h_density, D.data(), D.size() * sizeof(float));
    } catch (...) {
        return RADON_ENOMEM;
    }
    return RADON_OK;
}

// ---- polynomial sinogram filter and the solver iteration -------------
static int filter_setup(radon_plan *p, int order)
{
    if (order < 0 || order >= FILTER_MAXQ) return RADON_EINVAL;
    if (p->filter_order == order && p->filter_q[0] && p->filter_q[1]) return RADON_OK;
    CUDA_TRY(cudaDeviceSynchronize());                    // kernels in flight may still read the old tables
    cudaFree(p->filter_q[0]); cudaFree(p->filter_q[1]);
    p->filter_q[0] = p->filter_q[1] = nullptr;
    p->filter_order = -1;
    if (p->sgraph.exec) { cudaGraphExecDestroy(p->sgraph.exec); p->sgraph.exec = nullptr; }
    std::vector<float> q;
    int rc;
    try {
        build_filter_basis(p->dev.n_det, order, q);
        if ((rc = dev_upload(p, &p->filter_q[0], q))) return rc;
        build_filter_basis(p->dev.n_angles, order, q);
        if ((rc = dev_upload(p, &p->filter_q[1], q))) return rc;
    } catch (const std::bad_alloc &) {
        return RADON_ENOMEM;
    }
    p->filter_order = order;
    return RADON_OK;
}

extern "C" int radon_plan_set_filter(radon_plan *p, int order)
{
    if (!p) return RADON_EINVAL;
    return filter_setup(p, order);
}

extern "C" int radon_filter_basis_host(int n, int order, float *h_q)
{
    if (!h_q || n < 1 || order < 0 || order >= FILTER_MAXQ) return RADON_EINVAL;
    try {
        std::vector<float> q;
        build_filter_basis(n, order, q);
        for (int s = 0; s < n; ++s)
            for (int d = 0; d <= order; ++d) h_q[(size_t)s * (order + 1) + d] = q[(size_t)s * FILTER_MAXQ + d];
    } catch (...) {
        return RADON_ENOMEM;
    }
    return RADON_OK;
}

static int filter_ready(radon_plan *p) { return p->filter_order >= 0 ? RADON_OK : filter_setup(p, 3); }

extern "C" int radon_filter(radon_plan *p, const float *d_in, float *d_out, int axis, void *stream)
{
    if (!p || !d_in || !d_out || (axis != 0 && axis != 1)) return RADON_EINVAL;
    int rc = filter_ready(p);
    if (rc) return rc;
    if (launch_filter(p->dev, axis, p->filter_q[axis], p->filter_order, d_in, d_out, (cudaStream_t)stream)) return RADON_ECUDA;
    return check_launch();
}

// orders 0..3 run inside the projection DFT kernels; higher orders as a separate pass
extern "C" int radon_forward_filtered(radon_plan *p, const float *d_x, float *d_sino, void *stream)
{
    if (!p || !d_x || !d_sino) return RADON_EINVAL;
    int rc = filter_ready(p);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    ProjExtra ex;
    if (p->filter_order < FILTER_FUSED_Q) ex.q = p->filter_q[0];
    if ((rc = forward_ws(p, p->ws[0], d_x, d_sino, st, ex))) return rc;
    if (!ex.q && launch_filter(p->dev, 0, p->filter_q[0], p->filter_order, d_sino, d_sino, st)) return RADON_ECUDA;
    return check_launch();
}

static int resid_ready(radon_plan *p)
{
    return p->resid ? RADON_OK : dev_alloc(p, &p->resid, (size_t)p->M);
}

extern "C" int radon_adjoint_filtered(radon_plan *p, const float *d_sino, float *d_x, void *stream)
{
    if (!p || !d_x || !d_sino) return RADON_EINVAL;
    int rc = filter_ready(p);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (p->filter_order < FILTER_FUSED_Q) return adjoint_ws(p, p->ws[0], d_sino, d_x, st, nullptr, p->filter_q[0]);
    if ((rc = resid_ready(p))) return rc;
    if (launch_filter(p->dev, 0, p->filter_q[0], p->filter_order, d_sino, p->resid, st)) return RADON_ECUDA;
    return adjoint_ws(p, p->ws[0], p->resid, d_x, st);
}

// One iteration x <- S_tau(x - alpha Radon^T F (Radon x - b)), F the sinogram filter (filtered != 0)
// or the identity: the residual and the filter run in the epilogue of F4, the update and the
// shrinkage in the epilogue of A4; eight launches, no other kernels.
static int solver_step_on(radon_plan *p, float *d_x, const float *d_b, float alpha, float tau, int filtered, cudaStream_t st)
{
    ProjExtra ex;
    ex.sub = d_b;
    const bool fused = filtered && p->filter_order < FILTER_FUSED_Q;
    if (fused) ex.q = p->filter_q[0];
    int rc = forward_ws(p, p->ws[0], d_x, p->resid, st, ex);
    if (rc) return rc;
    if (filtered && !fused && launch_filter(p->dev, 0, p->filter_q[0], p->filter_order, p->resid, p->resid, st)) return RADON_ECUDA;
    IstaUpdate upd;
    upd.alpha = alpha; upd.tau = tau;
    return adjoint_ws(p, p->ws[0], p->resid, d_x, st, nullptr, nullptr, &upd);
}

extern "C" int radon_solver_step(radon_plan *p, float *d_x, const float *d_b, float alpha, float tau, int filtered, void *stream)
{
    if (!p || !d_x || !d_b || !(tau >= 0.f)) return RADON_EINVAL;
    int rc = resid_ready(p);
    if (rc) return rc;
    if (filtered && (rc = filter_ready(p))) return rc;
    return solver_step_on(p, d_x, d_b, alpha, tau, filtered, (cudaStream_t)stream);
}

// n_iter iterations: one iteration is captured once into a CUDA graph (on an internal stream: the
// caller's may be the legacy default stream, which cannot capture) and the graph is launched
// n_iter times on the caller's stream; it is re-captured when x, b, alpha, tau or the filter change.
extern "C" int radon_solver_run(radon_plan *p, float *d_x, const float *d_b, float alpha, float tau, int filtered,
                                int n_iter, void *stream)
{
    if (!p || !d_x || !d_b || !(tau >= 0.f) || n_iter < 0) return RADON_EINVAL;
    int rc = resid_ready(p);
    if (rc) return rc;
    if (filtered && (rc = filter_ready(p))) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (p->timer.enabled) {                               // stage events are not captured: run the plain calls
        for (int i = 0; i < n_iter && rc == RADON_OK; ++i) rc = solver_step_on(p, d_x, d_b, alpha, tau, filtered, st);
        return rc;
    }
    radon_plan::SolverGraph &g = p->sgraph;
    if (!g.exec || g.x != d_x || g.b != d_b || g.alpha != alpha || g.tau != tau || g.filtered != filtered) {
        if (g.exec) { cudaGraphExecDestroy(g.exec); g.exec = nullptr; }
        if (!p->capture_stream) CUDA_TRY(cudaStreamCreateWithFlags(&p->capture_stream, cudaStreamNonBlocking));
        CUDA_TRY(cudaStreamBeginCapture(p->capture_stream, cudaStreamCaptureModeThreadLocal));
        const long long n0 = launch_count();
        pdl_suppress(true);
        rc = solver_step_on(p, d_x, d_b, alpha, tau, filtered, p->capture_stream);
        pdl_suppress(false);
        g.kernels = launch_count() - n0;
        count_launch(-g.kernels);                       // captured, not launched
        cudaGraph_t graph = nullptr;
        cudaError_t e = cudaStreamEndCapture(p->capture_stream, &graph);
        if (rc == RADON_OK && e != cudaSuccess) {
            g_last_cuda_error = std::string("cudaStreamEndCapture: ") + cudaGetErrorString(e);
            rc = RADON_ECUDA;
        }
        if (rc == RADON_OK) {
            e = cudaGraphInstantiate(&g.exec, graph, 0);
            if (e != cudaSuccess) {
                g_last_cuda_error = std::string("cudaGraphInstantiate: ") + cudaGetErrorString(e);
                rc = RADON_ECUDA;
                g.exec = nullptr;
            }
        }
        if (graph) cudaGraphDestroy(graph);
        if (rc) return rc;
        g.x = d_x; g.b = d_b; g.alpha = alpha; g.tau = tau; g.filtered = filtered;
    }
    for (int i = 0; i < n_iter; ++i) CUDA_TRY(cudaGraphLaunch(g.exec, st));
    count_launch(g.kernels * n_iter);
    return RADON_OK;
}

// ---- batched device-pointer calls ------------------------------------------------------
// Slices are independent.  Consecutive slices go to BATCH_LANES internal streams
// with a workspace each, forked from and joined back into the caller's stream by events, so
// that the tail of one slice's kernel (most kernels leave part of the 148 SMs idle in their
// last wave) overlaps the head of the other slice's.  While stage timing is on the slices run
// one after the other on the caller's stream, so that the stage events mean what they say.
#ifndef RADON_BATCH_LANES
#define RADON_BATCH_LANES 4
#endif
constexpr int BATCH_LANES = RADON_BATCH_LANES;
static_assert(BATCH_LANES >= 1 && BATCH_LANES <= NWS, "one workspace per lane");

static int host_setup(radon_plan *p);

static int batch_run(radon_plan *p, bool fwd, const float *d_in, float *d_out, int batch, cudaStream_t user)
{
    if (!p || !d_in || !d_out || batch < 0) return RADON_EINVAL;
    const size_t nx = (size_t)p->dev.N * p->dev.N, ns = (size_t)p->M;
    const size_t n_in = fwd ? nx : ns, n_out = fwd ? ns : nx;
    const int lanes = (p->timer.enabled || batch < 2) ? 1 : BATCH_LANES;
    if (lanes == 1) {
        for (int b = 0; b < batch; ++b) {
            int rc = fwd ? forward_ws(p, p->ws[0], d_in + b * n_in, d_out + b * n_out, user)
                         : adjoint_ws(p, p->ws[0], d_in + b * n_in, d_out + b * n_out, user);
            if (rc) return rc;
        }
        return RADON_OK;
    }
    int rc = host_setup(p);                                 // streams, events, further workspaces
    if (rc) return rc;
    if (!p->fork_event) CUDA_TRY(cudaEventCreateWithFlags(&p->fork_event, cudaEventDisableTiming));
    CUDA_TRY(cudaEventRecord(p->fork_event, user));
    for (int l = 0; l < lanes; ++l) CUDA_TRY(cudaStreamWaitEvent(p->hstream[l], p->fork_event, 0));
    for (int b = 0; b < batch && rc == RADON_OK; ++b) {
        const int l = b % lanes;
        rc = fwd ? forward_ws(p, p->ws[l], d_in + b * n_in, d_out + b * n_out, p->hstream[l])
                 : adjoint_ws(p, p->ws[l], d_in + b * n_in, d_out + b * n_out, p->hstream[l]);
    }
    // join the lanes back into the caller's stream, also after a failure in the middle of the
    // fork (whatever was queued on the lanes stays ordered before the caller's next work)
    for (int l = 0; l < lanes; ++l) {
        cudaError_t e = cudaEventRecord(p->hevent[l], p->hstream[l]);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(user, p->hevent[l], 0);
        if (e != cudaSuccess && rc == RADON_OK) {
            g_last_cuda_error = std::string("batch join: ") + cudaGetErrorString(e);
            rc = RADON_ECUDA;
        }
    }
    return rc;
}

extern "C" int radon_forward_batch(radon_plan *p, const float *d_x, float *d_sino, int batch, void *stream)
{
    return batch_run(p, true, d_x, d_sino, batch, (cudaStream_t)stream);
}

extern "C" int radon_adjoint_batch(radon_plan *p, const float *d_sino, float *d_x, int batch, void *stream)
{
    return batch_run(p, false, d_sino, d_x, batch, (cudaStream_t)stream);
}

// ---- host-buffer entry points: NWS internal streams, copies of slice b+1 overlap kernels of slice b
static int host_setup(radon_plan *p)
{
    for (int i = 0; i < NWS; ++i) {
        if (!p->hstream[i]) CUDA_TRY(cudaStreamCreateWithFlags(&p->hstream[i], cudaStreamNonBlocking));
        if (!p->hevent[i]) CUDA_TRY(cudaEventCreateWithFlags(&p->hevent[i], cudaEventDisableTiming));
        int rc;
        if ((rc = workspace_alloc(p, p->ws[i]))) return rc;
        if (!p->ws[i].img && (rc = dev_alloc(p, &p->ws[i].img, (size_t)p->dev.N * p->dev.N))) return rc;
        if (!p->ws[i].sino && (rc = dev_alloc(p, &p->ws[i].sino, (size_t)p->M))) return rc;
    }
    return RADON_OK;
}

static int host_run(radon_plan *p, bool fwd, const float *h_in, float *h_out, int batch)
{
    if (!p || !h_in || !h_out || batch < 0) return RADON_EINVAL;
    int rc = host_setup(p);
    if (rc) return rc;
    // The internal streams share ws[0..] with device-pointer calls the caller may still have in
    // flight on a stream this call cannot see: order after everything queued on the device.
    // (The host entry points are synchronous anyway: they return after the last copy landed.)
    CUDA_TRY(cudaDeviceSynchronize());
    const size_t nx = (size_t)p->dev.N * p->dev.N, ns = (size_t)p->M;
    const size_t n_in = fwd ? nx : ns, n_out = fwd ? ns : nx;
    const int lanes = p->timer.enabled ? 1 : NWS;   // stage events mean something on one stream only
    for (int b = 0; b < batch; ++b) {
        const int i = b % lanes;
        cudaStream_t st = p->hstream[i];
        Workspace &w = p->ws[i];
        float *d_in = fwd ? w.img : w.sino, *d_out = fwd ? w.sino : w.img;
        CUDA_TRY(cudaMemcpyAsync(d_in, h_in + b * n_in, n_in * sizeof(float), cudaMemcpyHostToDevice, st));
        rc = fwd ? forward_ws(p, w, d_in, d_out, st) : adjoint_ws(p, w, d_in, d_out, st);
        if (rc) return rc;
        CUDA_TRY(cudaMemcpyAsync(h_out + b * n_out, d_out, n_out * sizeof(float), cudaMemcpyDeviceToHost, st));
    }
    for (int i = 0; i < NWS; ++i) CUDA_TRY(cudaStreamSynchronize(p->hstream[i]));
    return RADON_OK;
}

// x -> (Radon{x}, Radon^T{Radon{x}}) per slice: what a solver's normal-equation / gradient step needs.
// One upload (the image) and two downloads per slice, all on the slice's lane, so that the uploads
// of later slices run against the downloads of earlier ones (both PCIe directions busy at once).
extern "C" int radon_forward_adjoint_host(radon_plan *p, const float *h_x, float *h_sino, float *h_xt, int batch)
{
    if (!p || !h_x || !h_sino || !h_xt || batch < 0) return RADON_EINVAL;
    int rc = host_setup(p);
    if (rc) return rc;
    CUDA_TRY(cudaDeviceSynchronize());              // see host_run
    const size_t nx = (size_t)p->dev.N * p->dev.N, ns = (size_t)p->M;
    const int lanes = p->timer.enabled ? 1 : NWS;
    for (int b = 0; b < batch; ++b) {
        const int i = b % lanes;
        cudaStream_t st = p->hstream[i];
        Workspace &w = p->ws[i];
        CUDA_TRY(cudaMemcpyAsync(w.img, h_x + b * nx, nx * sizeof(float), cudaMemcpyHostToDevice, st));
        if ((rc = forward_ws(p, w, w.img, w.sino, st))) return rc;
        CUDA_TRY(cudaMemcpyAsync(h_sino + b * ns, w.sino, ns * sizeof(float), cudaMemcpyDeviceToHost, st));
        if ((rc = adjoint_ws(p, w, w.sino, w.img, st))) return rc;
        CUDA_TRY(cudaMemcpyAsync(h_xt + b * nx, w.img, nx * sizeof(float), cudaMemcpyDeviceToHost, st));
    }
    for (int i = 0; i < NWS; ++i) CUDA_TRY(cudaStreamSynchronize(p->hstream[i]));
    return RADON_OK;
}

extern "C" int radon_forward_host(radon_plan *p, const float *h_x, float *h_sino, int batch)
{
    return host_run(p, true, h_x, h_sino, batch);
}

extern "C" int radon_adjoint_host(radon_plan *p, const float *h_sino, float *h_x, int batch)
{
    return host_run(p, false, h_sino, h_x, batch);
}

// ---- test / measurement hooks ---------------------------------------------------------
extern "C" int radon_nufft2(radon_plan *p, const float *d_x, float *d_polar, void *stream)
{
    if (!p || !d_x || !d_polar) return RADON_EINVAL;
    int rc = nufft2_ws(p, p->ws[0], false, d_x, (float2 *)d_polar, (cudaStream_t)stream);
    mark(p, (cudaStream_t)stream, -1);
    return rc;
}

extern "C" int radon_nufft1(radon_plan *p, const float *d_polar, float *d_x, void *stream)
{
    if (!p || !d_x || !d_polar) return RADON_EINVAL;
    int rc = nufft1_ws(p, p->ws[0], false, (const float2 *)d_polar, d_x, (cudaStream_t)stream);
    mark(p, (cudaStream_t)stream, -1);
    return rc;
}

extern "C" int radon_interp_only(radon_plan *p, const float *d_grid, float *d_polar, void *stream)
{
    if (!p || !d_grid || !d_polar) return RADON_EINVAL;
    if (launch_gather(p->dev, false, (const float2 *)d_grid, (float2 *)d_polar, (cudaStream_t)stream)) return RADON_ECUDA;
    return check_launch();
}

extern "C" int radon_grid_only(radon_plan *p, const float *d_polar, float *d_grid, void *stream)
{
    if (!p || !d_grid || !d_polar) return RADON_EINVAL;
    if (launch_scatter(p->dev, false, (const float2 *)d_polar, (float2 *)d_grid, p->ws[0].scratch, p->ws[0].dcbuf, p->ws[0].tickets, (cudaStream_t)stream)) return RADON_ECUDA;
    return check_launch();
}

// ---- the paper's own gridding design, measured comparison ---------------------
extern "C" int radon_grid_only_paper_bins(radon_plan *p, const float *d_polar, float *d_grid, int n_bins, void *stream)
{
    if (!p || !d_polar || !d_grid || n_bins < 1) return RADON_EINVAL;
    if (!p->pb_bins || p->pb_target != n_bins) {
        CUDA_TRY(cudaDeviceSynchronize());
        cudaFree(p->pb_bins); cudaFree(p->pb_entries);
        p->pb_bins = nullptr; p->pb_entries = nullptr;
        PaperBins pb;
        try {
            build_paper_bins(p->geo, n_bins, pb);
        } catch (const std::bad_alloc &) {
            return RADON_ENOMEM;
        }
        int rc;
        if ((rc = dev_upload(p, &p->pb_bins, pb.bins))) return rc;
        if ((rc = dev_upload(p, &p->pb_entries, pb.entries))) return rc;
        p->pb_n_bins = (int)pb.bins.size(); p->pb_target = n_bins; p->pb_n_entries = (long long)pb.entries.size();
        p->pb_max_samples = 0; p->pb_unstaged = 0;
        for (const PaperBin &b : pb.bins) {
            p->pb_max_samples = std::max(p->pb_max_samples, b.count);
            p->pb_unstaged += b.count > 1024 ? 1 : 0;
        }
    }
    if (launch_paper_bins(p->dev, p->pb_bins, p->pb_n_bins, p->pb_entries, (const float2 *)d_polar, (float2 *)d_grid,
                          (cudaStream_t)stream)) return RADON_ECUDA;
    return check_launch();
}

extern "C" int radon_paper_bins_stats(const radon_plan *p, int *n_bins, long long *n_entries, int *max_samples, int *n_unstaged)
{
    if (!p || !p->pb_bins) return RADON_EINVAL;
    if (n_bins) *n_bins = p->pb_n_bins;
    if (n_entries) *n_entries = p->pb_n_entries;
    if (max_samples) *max_samples = p->pb_max_samples;
    if (n_unstaged) *n_unstaged = p->pb_unstaged;
    return RADON_OK;
}

extern "C" int radon_proj_ifft(radon_plan *p, const float *d_polar, float *d_sino, void *stream)
{
    if (!p || !d_polar || !d_sino) return RADON_EINVAL;
    if (launch_proj(true, false, p->dev, d_polar, d_sino, nullptr, (cudaStream_t)stream)) return RADON_ECUDA;
    return check_launch();
}

extern "C" int radon_proj_fft(radon_plan *p, const float *d_sino, float *d_polar, void *stream)
{
    if (!p || !d_polar || !d_sino) return RADON_EINVAL;
    if (launch_proj(false, false, p->dev, d_sino, d_polar, nullptr, (cudaStream_t)stream)) return RADON_ECUDA;
    return check_launch();
}

extern "C" int radon_plan_info(const radon_plan *p, int *N, int *G, int *n_angles, int *n_det,
                               long long *M, size_t *workspace_bytes)
{
    if (!p) return RADON_EINVAL;
    if (N) *N = p->dev.N;
    if (G) *G = p->dev.G;
    if (n_angles) *n_angles = p->dev.n_angles;
    if (n_det) *n_det = p->dev.n_det;
    if (M) *M = p->M;
    if (workspace_bytes) *workspace_bytes = p->device_bytes;
    return RADON_OK;
}

extern "C" int radon_plan_schedule_stats(const radon_plan *p, int half,
                                         long long *gather_slots, long long *gather_filled, int *gather_ctas,
                                         long long *scatter_slots, long long *scatter_filled, int *scatter_ctas)
{
    if (!p) return RADON_EINVAL;
    const int h = half ? 1 : 0;
    if (gather_slots) *gather_slots = p->gather_slots[h];
    if (gather_filled) *gather_filled = p->gather_filled[h];
    if (gather_ctas) *gather_ctas = p->dev.sched[h].n_gather_ctas;
    if (scatter_slots) *scatter_slots = p->scatter_slots[h];
    if (scatter_filled) *scatter_filled = p->scatter_filled[h];
    if (scatter_ctas) *scatter_ctas = p->dev.sched[h].n_scatter_ctas;
    return RADON_OK;
}

// Verifies the schedules the plan actually uses (device- or host-built): downloads the slot arrays
// and runs the host checker on them.
extern "C" int radon_plan_schedule_check(radon_plan *p, int half, long long *n_violations, int *device_built, double *build_ms)
{
    if (!p) return RADON_EINVAL;
    const int h = half ? 1 : 0;
    if (device_built) *device_built = p->device_built[h];
    if (build_ms) *build_ms = p->schedule_ms;
    if (!n_violations) return RADON_OK;
    *n_violations = -1;
    try {
        Schedules sch = p->meta[h];
        sch.gather_slots.resize((size_t)p->gather_slots[h]);
        sch.scatter_slots.resize((size_t)p->scatter_slots[h]);
        CUDA_TRY(cudaDeviceSynchronize());
        if (!sch.gather_slots.empty())
            CUDA_TRY(cudaMemcpy(sch.gather_slots.data(), p->dev.sched[h].gather_slots, sch.gather_slots.size() * sizeof(Slot), cudaMemcpyDeviceToHost));
        if (!sch.scatter_slots.empty())
            CUDA_TRY(cudaMemcpy(sch.scatter_slots.data(), p->dev.sched[h].scatter_slots, sch.scatter_slots.size() * sizeof(Slot), cudaMemcpyDeviceToHost));
        *n_violations = check_schedules(p->geo, sch);
        return *n_violations == 0 ? RADON_OK : RADON_EINVAL;
    } catch (const std::bad_alloc &) {
        return RADON_ENOMEM;
    }
}

extern "C" int radon_schedule_selfcheck(int N, int n_angles, int n_det, float sigma, int W, int half,
                                        long long *n_violations)
{
    if (n_violations) *n_violations = -1;
    int G = 0;
    int rc = validate(N, n_angles, n_det, sigma, W, &G);
    if (rc) return rc;
    try {
        Geometry geo;
        geo.init(N, n_angles, n_det, (double)sigma, W);
        Schedules sch;
        build_schedules(geo, sch, half != 0);
        const long long bad = check_schedules(geo, sch);
        if (n_violations) *n_violations = bad;
        return bad == 0 ? RADON_OK : RADON_EINVAL;
    } catch (...) {
        return RADON_ENOMEM;
    }
}

extern "C" int radon_schedule_host_stats(int N, int n_angles, int n_det, float sigma, int W, int half,
                                         long long out[10])
{
    if (!out) return RADON_EINVAL;
    int G = 0;
    int rc = validate(N, n_angles, n_det, sigma, W, &G);
    if (rc) return rc;
    try {
        Geometry geo;
        geo.init(N, n_angles, n_det, (double)sigma, W);
        Schedules sch;
        build_schedules(geo, sch, half != 0);
        long long mg = 0, ms = 0;
        for (const auto &c : sch.gather_ctas) mg = std::max<long long>(mg, c.round_count);
        for (const auto &c : sch.scatter_ctas)
            for (const auto &it : c.items) ms = std::max<long long>(ms, it.round_count);
        out[0] = (long long)sch.gather_slots.size(); out[1] = sch.gather_filled;
        out[2] = (long long)sch.gather_ctas.size(); out[3] = mg;
        out[4] = (long long)sch.scatter_slots.size(); out[5] = sch.scatter_filled;
        out[6] = (long long)sch.scatter_ctas.size(); out[7] = ms;
        out[8] = (long long)sch.merge_jobs.size(); out[9] = sch.n_partial_slots;
        return RADON_OK;
    } catch (...) {
        return RADON_ENOMEM;
    }
}

extern "C" int radon_kb_weights_host(int W, float sigma, float delta, float *w)
{
    if (!w || W < 2 || W > 12 || !(sigma > 1.0f) || !(delta >= 0.f && delta <= 1.f)) return RADON_EINVAL;
    if (!kw_supported(W)) return RADON_EUNSUPPORTED;
    KbPoly kp;
    build_kb_poly(W, sigma, kp);
    RADON_FOR_W(W, {
        float tmp[WW];
        kb_poly_weights<WW>(kp, delta, tmp);
        for (int l = 0; l < WW; ++l) w[l] = tmp[l];
    })
    return RADON_OK;
}

// ---- gridding without any allocation: scratch in a file-scope device array ---------------------
// radon_grid_only_static runs the scatter kernel of radon_grid_only with its scratch (partial
// rectangles of split tiles, merge counters, the summed j = 0 samples) in the three arrays below
// instead of a plan workspace, for callers that cannot call cudaMalloc (a stream under graph capture,
// a tight serving loop, a harness that forbids allocation).  Every GPU that loads the library holds
// the arrays (32 MiB + 32 KiB + 648 B) until the process exits.  In host code the array names are
// host-side stand-ins, not device addresses: their device addresses are resolved once per device,
// with that device current, by cudaGetSymbolAddress (static_scratch_of) and passed to the kernel.
// All calls on a device share the arrays: two calls that overlap on the GPU race.
constexpr int STATIC_SCRATCH_SLOTS = RADON_STATIC_SCRATCH_SLOTS;   // partial rectangles of SR_X x SR_Y cells (16 KiB each)
constexpr int STATIC_SCRATCH_JOBS = RADON_STATIC_SCRATCH_JOBS;     // merge jobs (MERGE_COUNTERS_PER_JOB counters each)
static __device__ __align__(256) float2 g_static_scratch[(size_t)STATIC_SCRATCH_SLOTS * SR_X * SR_Y];
static __device__ __align__(256) int g_static_tickets[STATIC_SCRATCH_JOBS * MERGE_COUNTERS_PER_JOB];
static __device__ __align__(256) float2 g_static_dcbuf[(KW_MAX + 1) * (KW_MAX + 1)];

struct StaticScratch { float2 *scratch = nullptr; int *tickets = nullptr; float2 *dcbuf = nullptr; bool ready = false; };
constexpr int STATIC_MAX_DEVICES = 64;
static StaticScratch g_static_dev[STATIC_MAX_DEVICES];
static std::mutex g_static_mutex;

// device addresses of the arrays on the current device (resolved at the first call on that device)
static int static_scratch_of(StaticScratch &out)
{
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) { g_last_cuda_error = "radon_grid_only_static: device ordinal above 63"; return RADON_ECUDA; }
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticScratch &d = g_static_dev[dev];
    if (!d.ready) {
        CUDA_TRY(cudaGetSymbolAddress((void **)&d.scratch, g_static_scratch));
        CUDA_TRY(cudaGetSymbolAddress((void **)&d.tickets, g_static_tickets));
        CUDA_TRY(cudaGetSymbolAddress((void **)&d.dcbuf, g_static_dcbuf));
        d.ready = true;
    }
    out = d;
    return RADON_OK;
}

extern "C" int radon_grid_only_static(radon_plan *p, const float *d_polar, float *d_grid, void *stream)
{
    if (!p || !d_grid || !d_polar) return RADON_EINVAL;
    const DevicePlan::Sched &q = p->dev.sched[0];                 // the full-grid schedule, as radon_grid_only
    // a partial rectangle of a plan with tall tiles (Geometry::st_y) takes more than one 64 x 32 slot of the array
    if ((size_t)p->n_partial * SR_X * p->geo.sr_y() > (size_t)STATIC_SCRATCH_SLOTS * SR_X * SR_Y ||
        q.n_merge_jobs > STATIC_SCRATCH_JOBS) return RADON_ELIMIT;
    StaticScratch s;
    int rc = static_scratch_of(s);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    // the arrays keep the last call's contents.  The merge counters must start at zero (a launch
    // leaves them at zero, but a call that failed or was cut short need not have): cleared here, on
    // the caller's stream.  Partial rectangles and the j = 0 sum are written in full by the launch
    // before it reads them.
    if (q.n_merge_jobs > 0)
        CUDA_TRY(cudaMemsetAsync(s.tickets, 0, sizeof(int) * MERGE_COUNTERS_PER_JOB * (size_t)q.n_merge_jobs, st));
    if (launch_scatter(p->dev, false, (const float2 *)d_polar, (float2 *)d_grid, s.scratch, s.dcbuf, s.tickets, st)) return RADON_ECUDA;
    return check_launch();
}

extern "C" long long radon_kernel_launch_count(void) { return launch_count(); }

extern "C" const char *radon_strerror(int code)
{
    switch (code) {
    case RADON_OK: return "ok";
    case RADON_EINVAL: return "invalid argument";
    case RADON_ENOMEM: return "out of memory";
    case RADON_ECUDA: return "CUDA runtime error (see radon_last_cuda_error)";
    case RADON_EARCH: return "device is not compute capability 10.x (sm_100a build, no fallback)";
    case RADON_ELIMIT: return "the plan's gridding needs more scratch than the library's static arrays hold (radon_grid_only_static: 2048 partial rectangles, 2048 merge jobs; use radon_grid_only)";
    case RADON_EUNSUPPORTED: return "valid request outside this build (W not 4, 6 or 8, or sigma*N neither a power of two in [16, 8192] nor 3 or 5 times a power of two in [16, 2048], or n_det > 8192 (power of two) / 2*n_det-1 > 8192 (otherwise))";
    default: return "unknown error";
    }
}

extern "C" const char *radon_last_cuda_error(void) { return g_last_cuda_error.c_str(); }
