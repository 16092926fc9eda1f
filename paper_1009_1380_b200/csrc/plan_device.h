// plan_device.h -- device-side schedule construction (plan_device.cu), internal.
#pragma once
#include <vector>
#include <cuda_runtime.h>

#include "radon_internal.h"

namespace radon {

struct PackRegion {             // a grid tile whose candidate samples are enumerated
    int rx0, ry0, rw, rh;       // cells (scatter: absolute; gather: after the row shift `oy`)
    int lo;                     // W - 1: every footprint that touches the tile (scatter); 0: base cell inside (gather)
    int oy;                     // row shift of the gather's tile grid (Hermitian half), else 0
    int n_in, n_cl;             // device: candidates wholly inside / clipped by the tile
    int K;                      // host: lists the tile's candidates are dealt to
    int max_row;                // device: most candidates on one base row (they can share a round only W apart)
};

struct PackList {               // one gather tile, or one of the K shares of a scatter tile
    int region, kk, K, n;
    long long cand_begin;       // candidate scratch
    long long tmp_round_begin;  // round scratch (round_cap rounds)
    long long round_begin;      // final place of its rounds
    int round_cap;
    int n_rounds, n_fast, filled, overflow;     // device results
    int pad;
    const Slot *src;            // its rounds in the round scratch of the attempt that packed it
};

struct DevicePackParams {
    int n_angles, n_det, G, W;
    int k0, k1, skip_k;         // samples k in [k0, k1) except skip_k
    int pitch;                  // shared-memory row pitch (complex) the bank pairs are computed for
    bool disjoint;              // scatter: footprints of a round must not meet within a row step
    void (*split)(std::vector<PackRegion> &, void *);   // sets K of every region from its counts
    // after an attempt: regions (indices) to deal to more lists and pack again, their K already raised
    void (*redo)(std::vector<PackRegion> &, const std::vector<PackList> &, int attempt, void *, std::vector<int> &);
    void *split_arg;
};

// Counts, fills and packs on the current device.  regions: in/out (counts, K); lists: out.
// *d_slots_out: cudaMalloc'ed array of 32 * *n_rounds_out slots (owned by the caller).
// Returns 0, -1 (CUDA error) or -2 (a list outgrew its round scratch: use the host builder).
int device_pack(const double2 *d_cs, const DevicePackParams &prm, std::vector<PackRegion> &regions,
                std::vector<PackList> &lists, Slot **d_slots_out, long long *n_rounds_out);

// Both schedules of a plan half built on the device.  out: everything except the slot arrays,
// which stay on the device (*d_gather_slots, *d_scatter_slots; out.gather_slots / scatter_slots
// are left empty).  Same return codes as device_pack.
int build_schedules_device(const Geometry &g, const double2 *d_cs, bool half, int n_workers, Schedules &out,
                           Slot **d_gather_slots, long long *n_gather_rounds,
                           Slot **d_scatter_slots, long long *n_scatter_rounds);

// Density compensation D of PAPER.md:89 times `scale`, one thread per sample (plan_device.cu); and the
// pair mean the Hermitian-half scatter needs for even n_det (in place).
int launch_density(const double2 *d_cs, int n_angles, int n_det, int W, double beta, double inv_i0b, double scale,
                   float *d_D, cudaStream_t st);
int launch_density_pair_mean(float *d_D, int n_angles, int n_det, cudaStream_t st);

}  // namespace radon
