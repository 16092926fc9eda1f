/*
 * radon.h -- C ABI of libradon_b200: the gridding / inverse-gridding (NUFFT)
 * pair behind the fast Radon transform y = Radon{x} and its adjoint, hand-written
 * CUDA for NVIDIA B200 (sm_100a).
 *
 * Source of the operations: Maia et al., "Compressive Phase Contrast Tomography",
 * arXiv 1009.1380.  "PAPER.md:NN" cites a line of the reference text.
 *
 *   - the solver "requires us to provide a function to perform y = Radon{x}"
 *     (section I) -> radon_forward; the solver also applies the
 *     transpose every iteration -> radon_adjoint.
 *   - "first perform a 2D FFT of x on a regular grid, and then interpolate the
 *     transform onto a polar grid before 1D inverse Fourier transforms are applied
 *     to interpolated points along the same radial lines" (section II)
 *     -> the stages of radon_forward; radon_adjoint runs the transposed stages in
 *     reverse order.
 *   - "The gridding operation requires the convolution between irregular samples
 *     and a kernel calculated at regular sample position and vice versa"
 *      with the sums printed beside Fig. 5:
 *       G_i(x_i,y_i) = sum_r G_r(x_r,y_r) K(x_r-x_i, y_r-y_i)
 *         -> radon_interp_only  (inverse gridding, regular -> polar, a gather)
 *       G_r(x_r,y_r) = sum_i D G(x_i,y_i) K(x_i-x_r, y_i-y_r)   (D == 1)
 *         -> radon_grid_only    (gridding, polar -> regular, a scatter)
 *   - the paper names neither kernel nor oversampling; BASELINE.json north_star
 *     fixes a Kaiser-Bessel kernel of width W = 6 on a sigma = 2 oversampled grid.
 *
 * Conventions (DESIGN.md section 4 lists every reading of the paper):
 *   image     x[iy*N + ix], fp32, row-major; centred coordinates X = ix - N/2,
 *             Y = iy - N/2 (integer division).
 *   sinogram  y[a*n_det + s], fp32, angle-major; theta_a = pi*a/n_angles,
 *             detector coordinate t = s - n_det/2 = X cos(theta) + Y sin(theta).
 *   polar     P[a*n_det + k], complex64 stored as interleaved (re, im) floats;
 *             radial frequency index j = k - n_det/2, sample position on the
 *             oversampled grid kappa = (G j / n_det)(cos theta_a, sin theta_a).
 *   grid      g[cy*G + cx], complex64 interleaved, G = sigma*N, CENTRED layout:
 *             cell (cx, cy) holds frequency (cx - G/2, cy - G/2); indices wrap
 *             mod G (the DTFT is periodic).
 *   Operator  S[a,s] = Re{ (1/n) sum_k F[a,k] exp(+i 2 pi j t/n) },
 *             F[a,k] = sum_pix x exp(-i (2 pi j/n)(X cos + Y sin));
 *             radon_adjoint is its exact transpose (no density weights, no 1/M).
 *
 * Pointers: every d_* argument is a DEVICE pointer owned by the caller (e.g. a
 * torch tensor's data_ptr()); every h_* argument is a HOST pointer owned by the
 * caller.  `stream` is a cudaStream_t passed as void* (NULL = default stream).
 * Device entry points are asynchronous on `stream`; input and output must not
 * alias.  A plan owns its tables and workspace, belongs to the CUDA device that
 * was current at creation, and must not be used from two streams at once.
 *
 * Errors: every call returns RADON_OK (0) or a negative code; nothing throws.
 * There is no CPU fallback and no other backend: on a machine without an sm_100
 * device radon_plan_create returns RADON_EARCH / RADON_ECUDA.
 */
#ifndef RADON_B200_H
#define RADON_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RADON_OK            0
#define RADON_EINVAL       -1   /* bad argument (see each call) */
#define RADON_ENOMEM       -2   /* host or device allocation failed */
#define RADON_ECUDA        -3   /* a CUDA runtime call failed (radon_last_cuda_error) */
#define RADON_EARCH        -4   /* current device is not compute capability 10.x */
#define RADON_ELIMIT       -6   /* radon_grid_only_static: the plan needs more scratch than the static arrays hold */
#define RADON_EUNSUPPORTED -5   /* valid but not built: W not 4, 6 or 8; sigma*N neither a power of two in [16, 8192]
                                   nor 3 or 5 times a power of two in [16, 2048];
                                   n_det > 8192 (power of two) or 2*n_det - 1 > 8192 (otherwise) */

typedef struct radon_plan radon_plan;   /* opaque, owned by the library */

/* Plan for images N x N, n_angles uniform angles in [0, pi), n_det detector bins,
 * oversampling sigma (G = sigma*N must be an even integer; this build takes a power of two,
 * 16 <= G <= 8192 -- the tuned FFT passes -- or 3 or 5 times a power of two in [16, 2048], e.g. N = 1536
 * or 2560 at sigma = 2 -- plainer passes, about 1.6 times the time per grid cell) and Kaiser-Bessel width W (this build: 4, 6 or 8; the gridding
 * kernels are instantiated for each; 6 is north_star's and the one the benchmarks run).
 * Builds, for the current CUDA device: per-angle fp64 direction table (Fourier
 * slice geometry), Kaiser-Bessel weight table (polynomial pieces) and de-apodisation vectors,
 * the conflict-free gather/scatter schedules (the plan-time binning that takes
 * the place of the paper's load-balanced bins), FFT twiddles and
 * chirp tables, and the workspace.  EINVAL: N < 8, n_angles < 1, n_det < 2,
 * n_angles > 65535 or n_det > 65533, sigma*N not an even integer, sigma outside (1, 8],
 * W outside [2,12], out == NULL.  EUNSUPPORTED: see above.  On failure *out is set to NULL.
 * Device memory: one workspace (T + grid + polar, 185 MB at N = 2048) at creation; the batched
 * and host-buffer calls allocate three more on first use (four slices in flight). */
int radon_plan_create(radon_plan **out, int N, int n_angles, int n_det, float sigma, int W);

/* Frees everything the plan owns (synchronises the device first). NULL is OK. */
int radon_plan_destroy(radon_plan *p);

/* y = Radon{x}.  d_x: N*N fp32.  d_sino: n_angles*n_det fp32. */
int radon_forward(radon_plan *p, const float *d_x, float *d_sino, void *stream);

/* x~ = Radon^T{y}: exact transpose of radon_forward (PAPER.md:85 with D == 1). */
int radon_adjoint(radon_plan *p, const float *d_sino, float *d_x, void *stream);

/* `batch` contiguous slices sharing the plan (BASELINE.json configs[4]).  The slices run on
 * four internal streams forked from and joined into `stream` (asynchronous for the caller
 * exactly like the single-slice calls); while stage timing is enabled they run one by one. */
int radon_forward_batch(radon_plan *p, const float *d_x, float *d_sino, int batch, void *stream);
int radon_adjoint_batch(radon_plan *p, const float *d_sino, float *d_x, int batch, void *stream);

/* Same operators on HOST buffers (pinned or pageable): slices are copied to the
 * device, transformed and copied back on four internal streams (one workspace each) so
 * that the copies of neighbouring slices overlap the kernels.  Synchronous on both
 * sides: the call first waits for everything queued on the device (cudaDeviceSynchronize:
 * device-pointer calls of this plan still in flight on a caller stream share its workspace)
 * and returns after the last copy has landed.  While stage timing is enabled the slices
 * run one by one on a single internal stream.
 * h_x: batch*N*N fp32, h_sino: batch*n_angles*n_det fp32. */
int radon_forward_host(radon_plan *p, const float *h_x, float *h_sino, int batch);
int radon_adjoint_host(radon_plan *p, const float *h_sino, float *h_x, int batch);

/* Both operators in one call, per slice: h_sino = Radon{h_x} and h_xt = Radon^T{h_sino} (the product
 * a solver's gradient step needs).  The sinogram is not uploaded again, and because every slice has
 * one upload and two downloads on its own lane, uploads and downloads of neighbouring slices use
 * both PCIe directions at once.  Synchronous like the calls above.  h_xt: batch*N*N fp32. */
int radon_forward_adjoint_host(radon_plan *p, const float *h_x, float *h_sino, float *h_xt, int batch);

/* Bare NUFFT (type 2): image -> M = n_angles*n_det complex polar samples
 * F[a,k] (de-apodise + zero-pad, 2-D FFT, inverse gridding).  d_polar: 2*M floats. */
int radon_nufft2(radon_plan *p, const float *d_x, float *d_polar, void *stream);
/* Its transpose on arbitrary complex polar input; output is the real part
 * (gridding, 2-D inverse FFT, crop + de-apodise).  d_x: N*N fp32. */
int radon_nufft1(radon_plan *p, const float *d_polar, float *d_x, void *stream);

/* Inverse gridding alone: d_grid 2*G*G floats (centred layout)
 * -> d_polar 2*M floats. */
int radon_interp_only(radon_plan *p, const float *d_grid, float *d_polar, void *stream);
/* Gridding alone (D == 1): d_polar 2*M floats -> d_grid 2*G*G floats;
 * every cell of d_grid is written exactly once (zeros included), no atomics, and
 * the result is bit-identical from run to run. */
int radon_grid_only(radon_plan *p, const float *d_polar, float *d_grid, void *stream);

/* radon_grid_only for callers that cannot allocate (a stream under CUDA graph capture, a serving
 * loop, a harness that forbids cudaMalloc): same arguments, same kernel, same schedule, bit-identical
 * result, but the kernel's scratch -- the partial rectangles of tiles whose samples are dealt to
 * several thread blocks, the counters of their merge, the summed j = 0 samples -- lives in
 * file-scope device arrays of the library instead of a plan workspace.  The call allocates and
 * frees nothing (no cudaMalloc / cudaFree / allocating library routine): one cudaMemsetAsync of
 * the merge counters and one kernel launch on `stream`; at the first call on a device it also
 * resolves the arrays' device addresses (cudaGetSymbolAddress, no allocation) -- make that call
 * outside a capture.
 *   Limits: RADON_STATIC_SCRATCH_SLOTS partial rectangles (64 x 32 complex cells, 16 KiB each:
 * 32 MiB; plans with sigma*N >= 4096 use 64 x 40 tiles and take 1.25 slots per rectangle) and RADON_STATIC_SCRATCH_JOBS merge jobs.  Every GPU that loads the library holds these
 * arrays (32 MiB + 33 KiB) until the process exits.  BASELINE.json's configs need 64 to ~1500
 * rectangles; a plan that needs more than the limit (millions of samples on a small grid, e.g.
 * 1024^2 with 4096 x 2048 samples: ~5500 rectangles) is rejected with RADON_ELIMIT before anything
 * is launched; use radon_grid_only for it.
 *   The arrays are shared by every call on a device, whatever the plan or stream, and keep the
 * last call's contents: the counters are cleared by the call itself, everything else is written
 * by the launch before it is read.  Two calls that overlap on the GPU (different streams, or
 * graph branches) race on them: serialise such calls.
 * Errors: RADON_EINVAL (null argument), RADON_ELIMIT, RADON_ECUDA. */
#define RADON_STATIC_SCRATCH_SLOTS 2048
#define RADON_STATIC_SCRATCH_JOBS 2048
int radon_grid_only_static(radon_plan *p, const float *d_polar, float *d_grid, void *stream);

/* The paper's own GPU design for the same gridding sum, kept as a measured comparison (prior
 * art, not the product path): load-balanced bins by recursive four-way splitting of the most
 * expensive bin (cost = samples x grid points), one thread block per bin, one thread per grid
 * point over the samples staged in shared memory when they fit (<= 1024), all threads per grid
 * point otherwise.  n_bins: where the splitting stops; the bins are built on the
 * host at the first call with a given n_bins (blocking).  Same arguments, tap rule and weights
 * as radon_grid_only; the result differs by the order of the additions only. */
int radon_grid_only_paper_bins(radon_plan *p, const float *d_polar, float *d_grid, int n_bins, void *stream);
/* Bins of the last radon_grid_only_paper_bins call: count, sample incidences, samples of the
 * largest bin, bins whose samples do not fit in shared memory.  EINVAL before the first call. */
int radon_paper_bins_stats(const radon_plan *p, int *n_bins, long long *n_entries, int *max_samples, int *n_unstaged);

/* 1-D transforms along the projections alone (last step):
 * radon_proj_ifft: polar 2*M floats -> sinogram, S = Re{(1/n) sum_k P exp(+i 2 pi j t/n)};
 * radon_proj_fft:  sinogram -> polar, its transpose Yh = (1/n) sum_s y exp(-i 2 pi j t/n). */
int radon_proj_ifft(radon_plan *p, const float *d_polar, float *d_sino, void *stream);
int radon_proj_fft(radon_plan *p, const float *d_sino, float *d_polar, void *stream);

/* Stage timing (measurement only).  While enabled, radon_forward / radon_adjoint (and the
 * batch, host and nufft entry points) record one CUDA event on their stream at every stage
 * boundary (the event pool grows on demand; if an event cannot be created the sample is
 * truncated and radon_plan_stage_times reports RADON_ENOMEM once).
 * radon_plan_stage_times waits for the last recorded event, adds the elapsed device time of
 * every recorded stage to total_ms[stage] and its count to launches[stage], then clears the
 * pool.  Stages: 0 de-apodise+pad+column FFT, 1 row FFT, 2 inverse gridding (gather),
 * 3 projection inverse DFT, 4 projection DFT, 5 gridding (scatter + merge), 6 row inverse
 * FFT, 7 column inverse FFT + crop + de-apodise. */
int radon_plan_stage_timing(radon_plan *p, int enable);
int radon_plan_stage_times(radon_plan *p, double total_ms[8], long long launches[8]);

/* Any of the out pointers may be NULL.  workspace_bytes = device bytes the plan owns. */
int radon_plan_info(const radon_plan *p, int *N, int *G, int *n_angles, int *n_det,
                    long long *M, size_t *workspace_bytes);

/* ---- inverse Radon transform ("Fast Radon and inverse Radon transforms"; Fig. 5
 * equations :85 and :89) -------------------------------------------------------------------
 * x = scale * Re{ sum_{a,k} D[a,k] Yhat[a,k] exp(+i (2 pi j/n)(X cos theta_a + Y sin theta_a)) },
 * Yhat = the centred 1-D DFT of every projection (as in radon_adjoint), computed by gridding
 * (eq. :85) WITH the density compensation D(x_i,y_i) = 1 / sum_j K(x_i - x_j, y_i - y_j) of
 * eq. :89 (sum over all polar samples, K the Kaiser-Bessel kernel on the oversampled grid),
 * followed by the 2-D inverse FFT, crop and de-apodisation.  scale = n_det phihat(0)^2 / G^2
 * turns D into an area element of the Fourier plane.  D is a plan
 * constant, derived in fp64 by a CUDA kernel (one thread per sample) at the first call, which blocks
 * for it (tens of ms at 2048^2); radon_plan_prepare_inverse does that ahead of time.
 * d_sino: n_angles*n_det fp32 (device), d_x: N*N fp32 (device, written).  Asynchronous on
 * `stream` after the first call (from the first one after radon_plan_prepare_inverse, which also makes
 * it capturable in a CUDA graph).  Returns RADON_OK or a negative code as radon_adjoint. */
int radon_inverse(radon_plan *p, const float *d_sino, float *d_x, void *cuda_stream);
/* Builds the density table of radon_inverse now (blocking; no-op when it exists). */
int radon_plan_prepare_inverse(radon_plan *p);

/* D * scale as the plan uses it (M = n_angles*n_det floats, HOST pointer, may be NULL) and
 * scale (may be NULL).  Builds D if the plan has not done so yet. */
int radon_plan_density(radon_plan *p, float *h_density, double *scale);

/* The same table without a plan or a GPU (host only; used by the CPU tests). */
int radon_density_host(int N, int n_angles, int n_det, float sigma, int W, float *h_density, double *scale);

/* ---- the sinogram filter of the paper's objective and the solver iteration -------------------
 * "we employed a 3rd order polynomial fit to smooth the sinogram and reduce the ringing
 * artifacts"; the reconstruction solves min ||x||_1 subject to
 * ||filter(Radon{x} - data)||_2 < eps, "filter is a polynomial interpolation operator"
 * (PAPER.md:31, :47), applied as "polynomial subtraction".  Reading R-filter
 * (DESIGN.md section 4): along one axis of the sinogram the least-squares polynomial of degree
 * `order` is subtracted; the operator is an orthogonal projector (symmetric, idempotent).
 *
 * radon_plan_set_filter: order 0..7 (default 3, used when a filtered call comes first); builds the
 * orthonormal discrete polynomial bases (fp64 on the host) and uploads them; synchronises the
 * device.  EINVAL: order outside [0, 7]. */
int radon_plan_set_filter(radon_plan *p, int order);
/* d_out = filter(d_in), both n_angles*n_det fp32 (device; d_out may equal d_in).
 * axis 0: along the detector coordinate of every projection (the exposure-to-exposure
 * fluctuation of the illuminating beam); axis 1: along the angle coordinate of every
 * detector bin.  Asynchronous on `stream`.  EINVAL: null pointer, axis not 0 or 1. */
int radon_filter(radon_plan *p, const float *d_in, float *d_out, int axis, void *stream);
/* filter(Radon{x}) and Radon^T{filter(y)}, filter along the projections (axis 0): for orders up to
 * 3 the filter runs inside the projection DFT kernels (no extra pass over the sinogram). */
int radon_forward_filtered(radon_plan *p, const float *d_x, float *d_sino, void *stream);
int radon_adjoint_filtered(radon_plan *p, const float *d_sino, float *d_x, void *stream);
/* Host only, no GPU: the basis the kernels use, h_q[s*(order+1) + d] = q_d(s), s < n. */
int radon_filter_basis_host(int n, int order, float *h_q);

/* One iteration of iterative soft-thresholding on the paper's objective (the
 * solver "requires us to provide a function to perform y = Radon{x}" every iteration):
 *   x <- S_tau( x - alpha * Radon^T{ F( Radon{x} - b ) } ),  S_tau(v) = sign(v) max(|v| - tau, 0),
 * F = the sinogram filter along the projections (filtered != 0) or the identity.  d_x: N*N fp32,
 * read and overwritten in place; d_b: the data, n_angles*n_det fp32.  Eight kernel launches: the
 * residual and the filter run in the epilogue of the projection inverse DFT, the update and the
 * shrinkage in the epilogue of the last inverse FFT pass.  EINVAL: null pointer, tau < 0. */
int radon_solver_step(radon_plan *p, float *d_x, const float *d_b, float alpha, float tau, int filtered,
                      void *stream);
/* n_iter such iterations; one iteration is captured into a CUDA graph inside the library (again
 * whenever an argument changes) and launched n_iter times on `stream`. */
int radon_solver_run(radon_plan *p, float *d_x, const float *d_b, float alpha, float tau, int filtered,
                     int n_iter, void *stream);

/* A plan holds two schedule sets.  half = 0: every polar sample and the whole grid (arbitrary
 * complex data: radon_nufft2/1, radon_interp_only, radon_grid_only).  half = 1: the Hermitian
 * half used by radon_forward / radon_adjoint, whose image and sinogram are real: the polar
 * samples obey F[a,-j] = conj F[a,j] and the gridded spectrum G(-k) = conj G(k), so only the
 * samples j >= 0 (plus, for even n_det, the mirror image j = +n/2 of the unpaired j = -n/2) are
 * interpolated, and only the grid rows ky = 0 .. G/2 are gridded.
 *
 * Schedule statistics of a plan (all host data; out pointers may be NULL):
 * slots = 32 * rounds issued, filled = slots holding a sample, ctas = thread blocks
 * per launch, for the gather (interp) and the scatter (grid) kernels. */
int radon_plan_schedule_stats(const radon_plan *p, int half,
                              long long *gather_slots, long long *gather_filled, int *gather_ctas,
                              long long *scatter_slots, long long *scatter_filled, int *scatter_ctas);

/* The schedules a plan uses are built by CUDA kernels (sample binning into tiles from the
 * Fourier-slice geometry and first-fit packing into conflict-free rounds, one warp per tile share);
 * the host builder below stays as the checker and as the fallback (a list that outgrows its
 * scratch, or RADON_PLAN_BUILDER=host in the environment).  radon_plan_schedule_check downloads the
 * plan's slot arrays and runs the same verification as radon_schedule_selfcheck on them.
 * *n_violations (may be NULL: no check), *device_built (1 if kernels built this half's schedules),
 * *build_ms (host wall time of both schedule sets inside radon_plan_create). */
int radon_plan_schedule_check(radon_plan *p, int half, long long *n_violations, int *device_built, double *build_ms);

/* Host-only self-check of the plan-time schedule builder; needs NO GPU.  Builds
 * the gather and scatter schedules for the geometry and verifies that every
 * sample is issued exactly once by the gather, that the scatter issues every
 * (sample, wrap image, output rectangle) incidence exactly once, that no two
 * samples issued to one warp in the same round touch the same cell within a row
 * step (write-conflict freedom without atomics) and that at most two lanes of a
 * half-warp start in the same shared-memory bank pair.  Returns RADON_OK or
 * RADON_EINVAL; *n_violations (may be NULL) receives the number of violations. */
int radon_schedule_selfcheck(int N, int n_angles, int n_det, float sigma, int W, int half,
                             long long *n_violations);

/* Host-only statistics of the schedules for a geometry (no GPU, no plan needed):
 * out[0..9] = gather slots, gather filled, gather CTAs, max gather rounds per CTA,
 * scatter slots, scatter filled, scatter CTAs, max scatter rounds per warp,
 * merge jobs, partial rectangles. */
int radon_schedule_host_stats(int N, int n_angles, int n_det, float sigma, int W, int half, long long out[10]);

/* Host-only evaluation of the W Kaiser-Bessel tap weights exactly as the kernels compute
 * them (plan-time polynomial pieces, fp32 Horner): w[l] = phi(delta - W/2 + l), l = 0..W-1,
 * for the fractional offset delta in [0,1].  Needs no GPU; used by the CPU unit tests. */
int radon_kb_weights_host(int W, float sigma, float delta, float *w);

/* Number of kernels the library has launched in this process (monotonic). */
long long radon_kernel_launch_count(void);

const char *radon_strerror(int code);
/* Text of the last CUDA error seen by this library on the calling thread. */
const char *radon_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* RADON_B200_H */
