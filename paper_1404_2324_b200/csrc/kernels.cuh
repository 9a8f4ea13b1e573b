// Kernel declarations (definitions in kernels.cu); see each definition for the operator it implements.
#pragma once
#include "state.cuh"

namespace genga {

constexpr int KP_THREADS = 256;   // threads per block of the pair kernel
constexpr int KP_TI = 2;          // bodies i per thread (register tile)
constexpr int KP_MAXJ = 256;      // longest j-slice staged in shared memory
constexpr int KP_HCAP = 1024;     // per-block list of pairs inside the precheck sphere

__global__ void k_begin_map(DevState d);
__global__ void k_reset_counters(DevState d);
__global__ void k_rcrit(DevState d, double tau);
__global__ void k_kick_pairs(DevState d, int record);
__global__ void k_kick_apply(DevState d, double h, double *aout);
__global__ void k_tp_kick(DevState d, double h, int record, double *aout);
__global__ void k_kick_multi(DevState d, double h, int record, double *aout);
__global__ void k_momentum(DevState d, const double *vx, const double *vy, const double *vz);
__global__ void k_shift(DevState d, double *ax, double *ay, double *az, double f, int divide_by_total);
__global__ void k_shift_out(DevState d, const double *ix, const double *iy, const double *iz,
                            double *ox, double *oy, double *oz, double f, int divide_by_total);
__global__ void k_drift(DevState d, double h);
__global__ void k_drift_arrays(long long n, double mu, double h, double *x, double *v, int *status);
__global__ void k_confirm(DevState d, double h);
__global__ void k_label_init(DevState d);
__global__ void k_union(DevState d);
__global__ void k_flatten(DevState d);
__global__ void k_build_groups(DevState d);
__global__ void k_bs_warp(DevState d, double h);
__global__ void k_bs_block(DevState d, double h);
template <int TW> __global__ void k_tp_bs(DevState d, double h, int lo);
__global__ void k_bs_multi(DevState d, double h);
__global__ void k_energy(DevState d, double *out);
__global__ void k_export_labels(DevState d, int *out);
__global__ void k_fp64_probe(double *out, int iters);

}  // namespace genga
