// Device-side view of one context's workspace (passed by value to every kernel).
#pragma once
#include "bs.cuh"
#include "common.cuh"

namespace genga {

struct DevState {
    int mode;        // 0 massive, 1 test particles, 2 multi system
    int nm;          // massive bodies per system
    int ntot;        // all bodies
    int nsys;        // systems
    int np;          // padded array stride (>= ntot)
    int nmtot;       // massive bodies in total (nm, or nsys*nm in mode 2)
    double G, n1, n2, eps;
    double *m0;      // [nsys]
    double *n12;     // mode 2: [nsys][2] the n1, n2 of every system (L346-354: set individually), else nullptr
    // democratic state, SoA [np]
    double *x, *y, *z, *vx, *vy, *vz, *m, *radius;
    double *rc, *c9;             // critical radius, 9 rc^2 (precheck threshold squared, L142)
    double *x0, *y0, *z0, *vx0, *vy0, *vz0;   // state before the drift (Eq. 10 needs both ends)
    int npm;         // nm padded to 128
    double *psum;    // [nsys][4]: sum m V (x,y,z) of the massive bodies, and sum m; mode 1: [2][4], slot 1 = the closing Sun kick's
    double *rcprev;  // mode 1: critical radii of the massive bodies in the step before (k_tp_mid)
    int2 *cand, *enc;
    long long cap;
    int *cnt;        // device ints: see CI_* below
    int *label;      // [np] group label of massive bodies
    int *gstart, *gsize, *gmem;  // groups of massive bodies (mode 0/1): [npm]
    int *gorder;                 // group numbers by decreasing size: the Bulirsch-Stoer queue (mode 2: (system, member mask) per group)
    unsigned *gmask;             // mode 1: bit mask of the massive group of body i
    unsigned *tpmask;            // mode 1: per particle, massive bodies it meets
    int *tplist;                 // mode 1: particles with encounters in this substep
    long long *stat;             // CNT_* accumulators
    double *kb;                  // mode 0: packed records (x, y, z, G m) of the massive bodies, [npm], padding far away and massless: the j-tile k_kick stages with bulk copies
    int *hcw;                    // mode 0: high word of the squared precheck radius KK_WIDE2 rc^2 per body (-1 for padding), [npm]
    unsigned *khits;             // mode 0: hit masks of the last closing kick, [blocks][KK_THREADS] (S2', k_kick)
    double *kfar;                // mode 0: its sums over the far pairs, [blocks][KK_THREADS][6]
    int4 *bstrace;               // [BS_TRACE_CAP] one record per group integrated in the last map (bs_trace in kernels.cu)
    BsScratch bss;
    // ---- collisions, ejections, removal (L316-332, L336, L378-384); off unless genga_set_collisions switches them on
    int coll;                    // collisions are looked for between the Bulirsch-Stoer steps
    int nmin;                    // a system with fewer bodies left is stopped (0 = never)
    double rcut2, rcutsun2;      // squared ejection limits (0 = none)
    int *kind;                   // [np] 0 massive, 1 test particle, 2 removed
    double *spin;                // [3][np]
    double *U;                   // [nsys] internal energy of the collisions (L318-322)
    double *ev;                  // event records, GENGA_EV doubles each (include/genga.h)
    long long evcap;
    int2 *redo;                  // groups k_bs_generic integrates: (kind << 28 | id, member mask); kinds: 0 massive group, 1 particle, 2 multi-system group
    BsScratch genA, genB;        // its scratch: genA indexed like gmem (massive groups are disjoint), genB 64 entries per block
};

// indices into DevState::cnt
enum : int { CI_NCAND = 0, CI_NENC = 1, CI_NGROUPS = 2, CI_NTP = 3, CI_STATUS = 4, CI_NTP_PREV = 5,
             CI_NBIG = 6, CI_QBIG = 7, CI_NMIDEND = 8, CI_QSMALL = 9, CI_QWARP = 10, CI_QTP = 11, CI_NTRACE = 12, CI_S2PMISS = 13, CI_NREDO = 14, CI_NCAND_TP = 15, CI_COUNT = 16 };   // CI_NCAND_TP: particle candidates (counted, not listed: k_tp_front)
constexpr int GEN_BLOCKS = 64;        // blocks of k_bs_generic
constexpr int BS_TRACE_CAP = 4096;   // records of genga_bs_trace kept per map

__device__ __forceinline__ int system_of(const DevState &d, int i) { return d.mode == 2 ? i / d.nm : 0; }

}  // namespace genga
