// Kernel declarations (definitions in kernels.cu); see each definition for the operator it implements.
#pragma once
#include "state.cuh"
#include "bs_cluster.cuh"
#include "bs_warp.cuh"
#include "multi_persist.cuh"

namespace genga {

constexpr int KK_THREADS = 896;   // threads per block of the kick kernel: 28 warps, 7 per SM sub-partition
constexpr int KK_WARPS = KK_THREADS / 32;
constexpr int KK_NI = 14;         // bodies i a block owns at most: ceil(2048 / 148)
constexpr int KK_MAXN = 2048;     // massive bodies of one system (L188)
// Squared radius of the kick's branch-free precheck in units of rc_ij^2: 3.3^2 instead of the 3^2 of the candidate test
// (L142).  The 10 % margin is what lets the opening kick of the NEXT step reuse the hit masks (S2', L266-274): its
// candidates r < 3 rc' are all hits as long as no critical radius grew by more than 10 % (k_rcrit checks).
constexpr double KK_WIDE2 = 10.89, KK_GROW = 1.0999;

// Bulirsch-Stoer layouts: groups of 2..8 bodies on one warp (bs_warp.cuh), of 9..256 bodies on a
// cluster of 8 CTAs (bs_cluster.cuh), larger ones on one block with a global-memory tableau (bs.cuh)
constexpr int BCB_MAXN = 256, BCB_THREADS = 256, BCB_LV = 2, BCB_CS = 8 * BCB_LV;   // BCB_LV trial step sizes side by side, 8 CTAs each

__global__ void k_begin_map(DevState d);
__global__ void k_reset_counters(DevState d);
__global__ void k_rcrit(DevState d, double tau, int reset, int check);
__global__ void k_kick(DevState d, double h, int record, int ni, double *aout, int to0, int s2p);
size_t kick_smem_bytes();
__global__ void k_tp_kick(DevState d, double h, int record, double *aout);
__global__ void k_tp_front(DevState d, double h, double tau, int first);
__global__ void k_tp_back(DevState d, double h);
__global__ void k_kick_multi(DevState d, double h, int record, double *aout);
__global__ void k_sun(DevState d, double h, int reset, double hdrift);
__global__ void k_multi_front(DevState d, double h, double hk);
__global__ void k_multi_back(DevState d, double h, double hk);
__global__ void k_coord_map(DevState d, const double *ix, const double *iy, const double *iz, double *ox, double *oy, double *oz, double f, int divide_by_total, int init);
__global__ void k_tiny_front(DevState d, double h, double tau, int first, double hk);
__global__ void k_tiny_back(DevState d, double h, double hk, int record, int reset);
__global__ void k_tpm_kick(DevState d, double h, int record, double fshift, int slot);
__global__ void k_tp_mid(DevState d, double hA, double hB, double tau, int newstep);
__global__ void k_momentum(DevState d, const double *vx, const double *vy, const double *vz, double fshift);
__global__ void k_shift(DevState d, double *ax, double *ay, double *az, double f, int divide_by_total);
__global__ void k_drift(DevState d, double h, double hsun);
__global__ void k_drift_arrays(long long n, double mu, double h, double *x, double *v, int *status);
__global__ void k_confirm(DevState d, double h);
__global__ void k_build_groups(DevState d);
template <int MAXN, int THREADS, int LV> __global__ void k_bs_cluster(DevState d, double h, int qslot, int endslot);
__global__ void k_bs_warp(DevState d, double h, int tp);
__global__ void k_list_groups_multi(DevState d);
__global__ void k_bs_block(DevState d, double h);
template <int TW> __global__ void k_tp_bs(DevState d, double h, int lo);
__global__ void k_tp_bs_big(DevState d, double h);
constexpr int TPBIG_BLOCKS = 16;   // blocks of k_tp_bs_big, 64 scratch entries each
__global__ void k_bs_multi(DevState d, double h);
__global__ void k_bs_generic(DevState d, double h, int pass);
__global__ void k_end_step(DevState d);
__global__ void k_end_step2(DevState d);
__global__ void k_energy(DevState d, double *out);
__global__ void k_export_labels(DevState d, int *out);
__global__ void k_fp64_probe(double *out, int iters);
__global__ void k_eval_fast(int which, long long n, const double *in, double *out);

}  // namespace genga
