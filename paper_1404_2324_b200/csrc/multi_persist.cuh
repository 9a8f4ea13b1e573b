// Multi-system mode, and massive mode with N <= 16 (one system: the paper's small-N regime, L427-433,
// where a step is launch latency): ALL the steps of a genga_step call in ONE launch, no grid-wide barrier.
//
// Systems never interact.  The launch-per-operator pipeline nevertheless made all 4096 systems of config 3 wait, in
// every map, for the one system that happened to be in a deep encounter (its Bulirsch-Stoer chain: ~45 us of a 110 us
// step).  Here a block of 128 threads holds 8 systems (16 lanes each, lane = body, padding lanes idle) with their state
// in shared memory and runs, for its own systems only, step after step: critical radii (Eq. 6), kick + precheck
// (Eq. 2), Sun kick (Eq. 3), Kepler drift (Eq. 9), encounter search (Eq. 10-12), grouping (connected components
// of 16 bodies as bit masks), Bulirsch-Stoer (the block layout of bs_small.cuh for groups of up to 8 bodies -- the
// whole block works on one group at a time --, the 16-lane team for larger ones), Sun kick, kick.  A block whose
// systems are quiet runs ahead; the launch lasts as long as the busiest block's own work, not the sum over the steps
// of every step's worst system.  Same arithmetic as the per-operator kernels: multi_pairs' pair loop, k_sun's sums in
// index order, kepler_drift, hermite_min, the Bulirsch-Stoer integrators.
// The candidate / encounter lists and labels genga_encounters returns are those of the last drift substep executed:
// written to global memory in the last map of the last step only.
#pragma once
#include "bs_small.cuh"
#include "state.cuh"

namespace genga {

constexpr int MP_SYS = 8, MP_LANES = 16, MP_THREADS = MP_SYS * MP_LANES;

struct MpSmem {
    double x[MP_THREADS], y[MP_THREADS], z[MP_THREADS], vx[MP_THREADS], vy[MP_THREADS], vz[MP_THREADS];
    double x0[MP_THREADS], y0[MP_THREADS], z0[MP_THREADS], vx0[MP_THREADS], vy0[MP_THREADS], vz0[MP_THREADS];
    double gm[MP_THREADS], rc[MP_THREADS], m[MP_THREADS];
    unsigned adj[MP_THREADS];            // encounter partners of a body (bits = lanes of its system)
    int2 groups[MP_THREADS / 2];         // (system of the block, member mask) of this map's groups
    int ngroups;
    BsmSmem W;
    TeamSmem<MP_LANES> team[MP_SYS];
};

// acceleration of body t by the bodies of its system (multi_pairs' arithmetic); cand = partners k > own lane inside the
// precheck sphere (L142)
__device__ __forceinline__ void mp_pairs(const MpSmem &S, int t, int sb, int nm, double xi, double yi, double zi, double rci,
                                         double &ax, double &ay, double &az, unsigned &cand)
{
    ax = ay = az = 0.0;
    cand = 0u;
    for (int k = 0; k < nm; ++k) {
        const int jt = sb + k;
        if (jt == t) continue;
        double dx = S.x[jt] - xi, dy = S.y[jt] - yi, dz = S.z[jt] - zi;
        double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
        double rcij = fmax(rci, S.rc[jt]);
        double gm = S.gm[jt];
        double s3 = gm * rinv3_fast(r2);
        if (r2 < 9.0 * rcij * rcij) {
            if (r2 < rcij * rcij) {                             // W = 1 outside the changeover zone
                double r = sqrt(r2);
                s3 = gm / (r2 * r) * kick_weight(r, rcij);
            }
            if (jt > t) cand |= 1u << k;
        }
        ax = fma(s3, dx, ax); ay = fma(s3, dy, ay); az = fma(s3, dz, az);
    }
}

__device__ __forceinline__ double rcrit_of(double G, double m0, double n1, double n2, double tau,
                                           double x, double y, double z, double vx, double vy, double vz, double m);

__global__ void __launch_bounds__(MP_THREADS) k_multi_persist(DevState d, double dt, int order, int nsteps)
#ifdef GENGA_KERNELS_CU
{
    __shared__ MpSmem S;
    const int t = threadIdx.x, nm = d.nm, sl = t / MP_LANES, k = t % MP_LANES, sb = sl * MP_LANES;
    const int sys = blockIdx.x * MP_SYS + sl;
    const bool live = sys < d.nsys && k < nm;
    const int i = sys * nm + k;                                  // global body index
    double w[7];
    const int nw = yoshida_weights(order, w);
    double x = 1e30 * (1 + t), y = 0.0, z = 0.0, vx = 0.0, vy = 0.0, vz = 0.0, m = 0.0, m0 = 1.0, n1 = 0.0, n2 = 0.0, rc = 0.0;
    if (live) {
        x = d.x[i]; y = d.y[i]; z = d.z[i]; vx = d.vx[i]; vy = d.vy[i]; vz = d.vz[i]; m = d.m[i];
        m0 = d.m0[sys];
        n1 = d.n12 ? d.n12[2 * sys] : d.n1; n2 = d.n12 ? d.n12[2 * sys + 1] : d.n2;      // per system (L346-354) / the one system of massive mode
    }
    S.m[t] = m; S.gm[t] = d.G * m;
    const double mu = d.G * m0;
    long long st_groups = 0, st_bs = 0, st_rej = 0, st_cand = 0;
    int st_max = 0;
    bool ok_kepler = true, ok_bs = true;
    unsigned cand = 0u;
#pragma unroll 1
    for (int step = 0; step < nsteps; ++step) {
        // ---- critical radii, once per step (Eq. 6)
        rc = live ? rcrit_of(d.G, m0, n1, n2, dt, x, y, z, vx, vy, vz, m) : 0.0;
        S.rc[t] = rc;
#pragma unroll 1
        for (int mp = 0; mp < nw; ++mp) {
            const double h = w[mp] * dt;
            const bool last_map = step == nsteps - 1 && mp == nw - 1;
            // ---- opening kick B(h/2) (first map of the step; later maps: done by the merged kick below)
            S.x[t] = x; S.y[t] = y; S.z[t] = z;
            __syncthreads();
            if (mp == 0) {
                double ax, ay, az;
                mp_pairs(S, t, sb, nm, x, y, z, rc, ax, ay, az, cand);
                if (live) { vx = fma(0.5 * h, ax, vx); vy = fma(0.5 * h, ay, vy); vz = fma(0.5 * h, az, vz); }
            }
            if (!live) cand = 0u;
            // ---- Sun kick C(h/2): s = sum m V of the own system, in index order (k_sun)
            S.vx[t] = vx; S.vy[t] = vy; S.vz[t] = vz;
            __syncthreads();
            {
                double sx = 0.0, sy = 0.0, sz = 0.0;
                for (int q = 0; q < nm; ++q) {
                    const double mq = S.m[sb + q];
                    sx = fma(mq, S.vx[sb + q], sx); sy = fma(mq, S.vy[sb + q], sy); sz = fma(mq, S.vz[sb + q], sz);
                }
                const double g = 0.5 * h / m0;
                x = fma(g, sx, x); y = fma(g, sy, y); z = fma(g, sz, z);
            }
            // ---- drift A(h), Kepler part; the state before it is kept (Eq. 10, Bulirsch-Stoer)
            S.x0[t] = x; S.y0[t] = y; S.z0[t] = z; S.vx0[t] = vx; S.vy0[t] = vy; S.vz0[t] = vz;
            if (live && !kepler_drift(mu, h, x, y, z, vx, vy, vz)) ok_kepler = false;
            __syncthreads();                                     // everybody has read the pre-kick positions
            S.x[t] = x; S.y[t] = y; S.z[t] = z; S.vx[t] = vx; S.vy[t] = vy; S.vz[t] = vz;
            S.adj[t] = 0u;
            __syncthreads();
            // ---- encounter search over my candidates (k_confirm's arithmetic)
            unsigned enc = 0u;
            for (unsigned cm = cand; cm; cm &= cm - 1) {
                const int q = __ffs(cm) - 1, jt = sb + q;
                double dx = S.x0[jt] - S.x0[t], dy = S.y0[jt] - S.y0[t], dz = S.z0[jt] - S.z0[t];
                double dvx = S.vx0[jt] - S.vx0[t], dvy = S.vy0[jt] - S.vy0[t], dvz = S.vz0[jt] - S.vz0[t];
                double P0 = dx * dx + dy * dy + dz * dz, Pd0 = 2.0 * (dx * dvx + dy * dvy + dz * dvz);
                dx = S.x[jt] - S.x[t]; dy = S.y[jt] - S.y[t]; dz = S.z[jt] - S.z[t];
                dvx = S.vx[jt] - S.vx[t]; dvy = S.vy[jt] - S.vy[t]; dvz = S.vz[jt] - S.vz[t];
                double P1 = dx * dx + dy * dy + dz * dz, Pd1 = 2.0 * (dx * dvx + dy * dvy + dz * dvz);
                const double rcij = fmax(S.rc[t], S.rc[jt]);
                if (hermite_min(P0, P1, Pd0, Pd1, h) < rcij * rcij) {
                    enc |= 1u << q;
                    atomicOr(&S.adj[jt], 1u << k);
                }
            }
            if (enc) atomicOr(&S.adj[t], enc);
            st_cand += __popc(cand);
            if (last_map && live) {                              // the lists genga_encounters returns
                if (cand) atomicAdd(&d.cnt[CI_NCAND], __popc(cand));
                for (unsigned em = enc; em; em &= em - 1) {
                    const int idx = atomicAdd(&d.cnt[CI_NENC], 1);
                    if (idx < d.cap) d.enc[idx] = make_int2(i, sys * nm + __ffs(em) - 1);
                    else atomicOr(&d.cnt[CI_STATUS], ERRBIT_CAPACITY);
                }
            }
            if (t == 0) S.ngroups = 0;
            __syncthreads();
            // ---- grouping: connected components of the <= 16 bodies of a system as bit masks (L537-565: label = lowest member)
            unsigned comp = S.adj[t] | (1u << k);
            if (__syncthreads_or(S.adj[t] != 0u)) {              // block-uniform: some system has an encounter
#pragma unroll 1
                for (int it = 0; it < 4; ++it) {                 // reach doubles: 4 rounds cover paths of 16 bodies
                    S.adj[t] = comp;
                    __syncthreads();
                    unsigned c2 = comp;
                    for (unsigned cm = comp; cm; cm &= cm - 1) c2 |= S.adj[sb + __ffs(cm) - 1];
                    __syncthreads();
                    comp = c2;
                }
                const bool root = live && (__ffs(comp) - 1) == k && __popc(comp) >= 2;
                if (root) { const int g = atomicAdd(&S.ngroups, 1); S.groups[g] = make_int2(sl, (int)comp); }
                __syncthreads();
                // a fixed order of the groups (the results do not depend on it; the trace and the counters do not either)
                const int ng = S.ngroups;
                // ---- Bulirsch-Stoer from the state before the drift, one group at a time by the whole block
#pragma unroll 1
                for (int g = 0; g < ng; ++g) {
                    const int2 gr = S.groups[g];
                    const unsigned mask = (unsigned)gr.y;
                    const int n = __popc(mask), gsb = gr.x * MP_LANES;
                    int nst[2] = {0, 0};
                    if (n <= BW_MAXN) {
                        const int lane = t & 31, b8 = lane & 7;
                        const int jt = b8 < n ? gsb + __fns(mask, 0, b8 + 1) : -1;
                        double Y[6] = {1.0, 0.0, 0.0, 0.0, 1.0, 0.0}, brc = 0.0, bm = 0.0;
                        if (jt >= 0) {
                            Y[0] = S.x0[jt]; Y[1] = S.y0[jt]; Y[2] = S.z0[jt]; Y[3] = S.vx0[jt]; Y[4] = S.vy0[jt]; Y[5] = S.vz0[jt];
                            brc = S.rc[jt]; bm = S.m[jt];
                        }
                        const double gm0 = d.G * d.m0[min(blockIdx.x * MP_SYS + gr.x, d.nsys - 1)];
                        if (t == 0) S.W.coll = 0;
                        int okg;
                        if (n <= 4) {
                            const int src = n == 2 ? (lane & 1) : (lane & 3);
#pragma unroll
                            for (int c = 0; c < 6; ++c) Y[c] = __shfl_sync(0xffffffffu, Y[c], src);
                            brc = __shfl_sync(0xffffffffu, brc, src); bm = __shfl_sync(0xffffffffu, bm, src);
                            if (n == 2) okg = bsm_integrate<2, BW_WARPS>(S.W, n, gm0, brc, bm, d.G, Y, h, d.eps, nst);
                            else okg = bsm_integrate<4, BW_WARPS>(S.W, n, gm0, brc, bm, d.G, Y, h, d.eps, nst);
                        } else okg = bsm_integrate<8, BW_WARPS>(S.W, n, gm0, brc, bm, d.G, Y, h, d.eps, nst);
                        if (!okg) ok_bs = false;
                        __syncthreads();
                        if (t < 8 && jt >= 0) { S.x[jt] = Y[0]; S.y[jt] = Y[1]; S.z[jt] = Y[2]; S.vx[jt] = Y[3]; S.vy[jt] = Y[4]; S.vz[jt] = Y[5]; }
                    } else if (sl == gr.x) {                     // more than 8 bodies: the system's own 16 lanes (bs.cuh)
                        const unsigned tmask = 0xffffu << ((t & 31) - k);
                        WarpTeam<MP_LANES> tm{tmask, k};
                        TeamSmem<MP_LANES> &T = S.team[sl];
                        const double trc = S.rc[t];
                        T.m[k] = S.m[t]; T.rc[k] = trc; T.irc[k] = trc > 0.0 ? 1.0 / (0.9 * trc) : 0.0;
                        tm.sync();
                        const bool active = (mask >> k) & 1u;
                        double q3[3] = {1.0, 0.0, 0.0}, V3[3] = {0.0, 1.0, 0.0};
                        if (active) { q3[0] = S.x0[t]; q3[1] = S.y0[t]; q3[2] = S.z0[t]; V3[0] = S.vx0[t]; V3[1] = S.vy0[t]; V3[2] = S.vz0[t]; }
                        if (!bs_team<MP_LANES>(tm, T, MP_LANES, active, mask, d.G, m0, trc, q3, V3, h, d.eps, nst)) ok_bs = false;
                        if (active) { S.x[t] = q3[0]; S.y[t] = q3[1]; S.z[t] = q3[2]; S.vx[t] = V3[0]; S.vy[t] = V3[1]; S.vz[t] = V3[2]; }
                    }
                    if (t == (n <= BW_MAXN ? 0 : gsb + __ffs(mask) - 1)) {
                        ++st_groups; st_bs += nst[0]; st_rej += nst[1]; st_max = max(st_max, n);
                    }
                    __syncthreads();
                }
                x = S.x[t]; y = S.y[t]; z = S.z[t]; vx = S.vx[t]; vy = S.vy[t]; vz = S.vz[t];
            }
            if (last_map && live) d.label[i] = sys * nm + __ffs(comp) - 1;
            // ---- Sun kick C(h/2) with the velocities after the drift / Bulirsch-Stoer
            {
                double sx = 0.0, sy = 0.0, sz = 0.0;
                for (int q = 0; q < nm; ++q) {
                    const double mq = S.m[sb + q];
                    sx = fma(mq, S.vx[sb + q], sx); sy = fma(mq, S.vy[sb + q], sy); sz = fma(mq, S.vz[sb + q], sz);
                }
                const double g = 0.5 * h / m0;
                x = fma(g, sx, x); y = fma(g, sy, y); z = fma(g, sz, z);
            }
            __syncthreads();                                     // the sums have been formed: positions may be overwritten
            // ---- closing kick B(h/2), merged with the opening kick of the next map of the same step (same positions, same
            // critical radii, R-4): one kick of (h + h_next)/2 that records the next map's candidates
            S.x[t] = x; S.y[t] = y; S.z[t] = z;
            __syncthreads();
            {
                const double hn = mp + 1 < nw ? w[mp + 1] * dt : 0.0;
                double ax, ay, az;
                unsigned c2;
                mp_pairs(S, t, sb, nm, x, y, z, rc, ax, ay, az, c2);
                const double hk = 0.5 * (h + hn);
                if (live) { vx = fma(hk, ax, vx); vy = fma(hk, ay, vy); vz = fma(hk, az, vz); }
                cand = c2;
            }
            __syncthreads();                                     // the pair loop has read the positions
        }
    }
    if (live) {
        d.x[i] = x; d.y[i] = y; d.z[i] = z; d.vx[i] = vx; d.vy[i] = vy; d.vz[i] = vz; d.rc[i] = rc; d.c9[i] = 9.0 * rc * rc;
    }
    if (!ok_kepler) atomicOr(&d.cnt[CI_STATUS], ERRBIT_KEPLER);
    if (!ok_bs) atomicOr(&d.cnt[CI_STATUS], ERRBIT_BS);
    if (st_groups) {
        atomicAdd((unsigned long long *)&d.stat[CNT_GROUPS], (unsigned long long)st_groups);
        atomicAdd((unsigned long long *)&d.stat[CNT_BSSTEPS], (unsigned long long)st_bs);
        atomicAdd((unsigned long long *)&d.stat[CNT_BSREJECTS], (unsigned long long)st_rej);
        atomicMax((unsigned long long *)&d.stat[CNT_MAXGROUP], (unsigned long long)st_max);
    }
    if (st_cand) atomicAdd((unsigned long long *)&d.stat[CNT_CAND], (unsigned long long)st_cand);
}
#else
;
#endif

}  // namespace genga
