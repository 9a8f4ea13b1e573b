// Bulirsch-Stoer for one close-encounter group on a thread-block CLUSTER.
//
// The cost of Bulirsch-Stoer on a GPU is latency, not arithmetic: one step is a chain of dependent force
// evaluations, and cfg1 has only ~165 groups per time step.  The paper parallelises inside one force evaluation
// (p threads per body, Table 3).  Here, in addition:
//   * the extrapolation COLUMNS run side by side: the modified-midpoint runs with n_k = 2, 4, ..., 16 substeps all
//     start from the same state, so CTA `col` of a level integrates column `col` (col + 1 double evaluations);
//   * LV trial step sizes H, H/2 (LEVELS) run side by side on 8 CTAs each (cluster of 8 LV CTAs): the level taken is
//     the first one, in that order, that passes -- the step the sequential rule ("first trial H; on failure H/2",
//     DESIGN.md R-7) arrives at after its rejections, so the accepted steps are the sequential algorithm's;
//   * EARLY EXIT: CTA 0 of a level has nothing to do after its one evaluation and becomes the level's CHECKER: as the
//     columns arrive (through distributed shared memory) it extends the Aitken-Neville tableau row by row and stops at
//     the first row whose error passes, exactly the row the sequential algorithm stops at.
// There is no cluster-wide barrier inside a step.  The master (CTA 0 of the cluster) publishes a record per round
// (round number, H, the state to start from) into the shared memory of every CTA under a sequence lock; a column CTA
// works on the round it finds, drops it as soon as a newer record appears (it looks once per evaluation), and signals
// its finished column with one remote flag store.  A CTA that lags simply joins the current round.
//
// Inside a CTA, thread i < n OWNS body i: it carries the body's midpoint state in registers, writes its positions to
// a double-buffered shared array before every force evaluation and adds up the forces on it afterwards (bc_rhs2); the
// other warps only evaluate pairs.  What an evaluation costs is the owners' dependent chain, counted in instructions
// (one warp per scheduler issues a dependent instruction every 5-9 cycles) and barriers (44 cycles each for 16 warps),
// and what a round costs beyond its evaluations is the master's own chain (its column, the tableau rows one after the
// other, the publication): both were measured with clock64 traces and shortened step by step (profiles/r2_bs_chain.md).
#pragma once
#include <cooperative_groups.h>

#include "bs.cuh"

namespace genga {

namespace cg = cooperative_groups;

constexpr int BC_MAXP = 768;         // entries of the pair table of bc_rhs2: (most partners of one body + 1) x (n | 1) must fit

template <int MAXN, int THREADS>
struct BcSmem {
    double pos[2][2][3][MAXN];      // [buffer][point A / B][component][body]
    float4 pf[2][2][MAXN];          // positions rounded to FP32 for the conservative pretest, .w = thr2: one LDS.128 per partner
    double isq[MAXN], isv[MAXN];    // checker: 1 / |q|^2, 1 / |V|^2 of the round's starting state (error norm)
    float thr2[MAXN];               // (rc_i + margin)^2 rounded up
    double m[MAXN], rc[MAXN], irc[MAXN];
    double R[MAXN];                 // physical radii (collision test; < 0: none)
    alignas(16) double Y[6][MAXN];  // state the current round starts from (pushed by the master)
    double tab[BS_KMAX][6][MAXN];   // checker: column results T[k][0] of its level
    double diag[6][MAXN];           // checker: T[k][k] of the row tested last
    double red[THREADS / 32];
    // ---- close pairs of the current evaluation (bc_rhs2, list path)
    int part[BC_MAXP];              // entry (k + 1) npad + i: the k-th partner of body i that passed the FP32 pretest at either point
    alignas(16) double pres[BC_MAXP][6];        // same entries: the acceleration of i by that partner at the two points; entry i (row 0): by the star
    int kmax[2];                    // most partners of one body (double-buffered like pos)
    int stale[2];                   // an owner found the list outdated (double-buffered like pos)
    int refbody;                    // the body nearest the group's centre
    int ok;                         // block-local broadcast: the record just read is consistent
    float4 ref[MAXN];               // positions (FP32) at the evaluation the list was built from
    int cnt[MAXN];                  // partners of body i in the list
    float skin2;                    // the list stays valid while every body has moved, in the central body's frame, by less than sqrt(skin2) (0: never)
    // ---- round record, written by the master under a sequence lock (seq_begin first, seq_end last).  Round numbers
    // run on from group to group, so a flag of an older round never equals a current one.
    volatile int seq_begin, seq_end;
    volatile double rec_H;          // the round's largest trial step (level l tries rec_H / 2^l)
    volatile int rec_state;         // 0 run the round, 1 group finished, 2 step size underflow, 3 a pair collides
    volatile int ready[BS_KMAX];    // checker: ready[k] = round whose column k has arrived
    volatile int lev_result[4];     // master: (round << 8) | code of level l; code 0 underflow, 1 rejected, 2 + k passed at row k
    int bc[2];                      // block-local broadcast of what thread 0 saw
    int cur;
};

struct BcLane {
    int n, L;
    int i;              // the body this thread OWNS (integrates, sums the forces of): thread i < n owns body i
    bool owner;
    int pi, s;          // lane s of the L lanes that examine the pairs of body pi (the n^2 distance tests)
};

// The list of close pairs the block carries from one evaluation to the next (bc_rhs2).
struct BcList {
    int rows, npad;     // S.part / S.pres: rows of npad entries (row 0 the star, row k + 1 the k-th partner of every body)
    unsigned magic;     // ceil(2^32 / npad): entry / npad without a division
    bool valid;
    int age;            // evaluations the current list has served
    double span, span_fail;   // time between this evaluation and the one before (set by the caller); the shortest one after
                        // which a list was found outdated at its first check: from there on (long trial steps, few
                        // substeps) a new list is made every time without trying the old one first
    int ref;            // the body the rigid motion is taken from: the one nearest the group's centre
};

#ifndef GENGA_BC_SKIN
#define GENGA_BC_SKIN 0.3
#endif
constexpr double BC_SKIN = GENGA_BC_SKIN;      // the list takes pairs out to (1 + BC_SKIN) rc_ij

template <int THREADS>
__device__ __forceinline__ BcLane bc_lanes(int n)
{
    int P = 2;
    while (P < n) P <<= 1;              // bodies, rounded up to a power of two
    BcLane t;
    t.n = n; t.L = min(8, THREADS / P);
    t.i = threadIdx.x; t.owner = threadIdx.x < n;
    t.pi = threadIdx.x / t.L; t.s = threadIdx.x % t.L;
    return t;
}

// The list path of bc_rhs2: one thread per entry of the table S.part (rows x npad; threads first, first + 1, ..,
// THREADS - 1 share them): row 0, column i the star's acceleration of body i; row k + 1, column i the acceleration of i by
// its k-th listed partner at the two points (zero where the pair is outside rc_ij).  Results go to the same entry of
// S.pres: npad is odd and an entry 48 bytes, so the LDS.128 of eight neighbouring owners walking down their columns fall
// into eight different groups of four banks (a compact list walked a lane every few entries measured 16-way conflicts:
// ~100 cycles per entry).
template <int MAXN, int THREADS>
__device__ __forceinline__ void bc_pairs(BcSmem<MAXN, THREADS> &S, const double (*pA)[MAXN], const double (*pB)[MAXN], double G, double m0,
                                         const BcList &lst, const int n, const int first)
{
    const int npad = lst.npad, entries = lst.rows * npad;
    for (int p = (int)threadIdx.x - first; p >= 0 && p < entries; p += THREADS - first) {
        const int row = (int)__umulhi((unsigned)p, lst.magic), i = p - row * npad;
        if (i >= n) continue;
        double *o = S.pres[p];
        if (row == 0) {
            const double xA = pA[0][i], yA = pA[1][i], zA = pA[2][i], xB = pB[0][i], yB = pB[1][i], zB = pB[2][i];
            const double sA = -G * m0 * rinv3_fast(xA * xA + yA * yA + zA * zA), sB = -G * m0 * rinv3_fast(xB * xB + yB * yB + zB * zB);
            *reinterpret_cast<double2 *>(o) = make_double2(sA * xA, sA * yA);
            *reinterpret_cast<double2 *>(o + 2) = make_double2(sA * zA, sB * xB);
            *reinterpret_cast<double2 *>(o + 4) = make_double2(sB * yB, sB * zB);
            continue;
        }
        if (row > S.cnt[i]) continue;
        const int j = S.part[p];
        const double rci = S.rc[i], rcj = S.rc[j];
        const bool big = rci >= rcj;
        const double rcij = big ? rci : rcj, rc2 = rcij * rcij;
        const double dx = pA[0][j] - pA[0][i], dy = pA[1][j] - pA[1][i], dz = pA[2][j] - pA[2][i];
        const double ex = pB[0][j] - pB[0][i], ey = pB[1][j] - pB[1][i], ez = pB[2][j] - pB[2][i];
        const double dA = dx * dx + dy * dy + dz * dz, dB = ex * ex + ey * ey + ez * ez;
        const bool inA = dA < rc2, inB = dB < rc2;
        const double ir = big ? S.irc[i] : S.irc[j];
        const double gmj = G * S.m[j];
        double wA = direct_scale_nb(inA ? dA : rc2, rcij, ir, gmj);
        double wB = direct_scale_nb(inB ? dB : rc2, rcij, ir, gmj);
        wA = inA ? wA : 0.0; wB = inB ? wB : 0.0;
        *reinterpret_cast<double2 *>(o) = make_double2(wA * dx, wA * dy);
        *reinterpret_cast<double2 *>(o + 2) = make_double2(wA * dz, wB * ex);
        *reinterpret_cast<double2 *>(o + 4) = make_double2(wB * ey, wB * ez);
    }
}

// Forces on body t.i at TWO sets of positions (qA, qB of the owners) at once (Eq. 1 L73-74 through Eq. 8
// L104; star fixed at the origin, L314; every pair of the group is examined at every evaluation, L505).
// Two at once because a(q_k) and a(q_{k+1}) of Gragg's rule are independent (bs_warp.cuh): one set of barriers
// serves both, and their dependent chains overlap.
//
// What an evaluation costs is latency and issue slots, not arithmetic (measured on B200, one warp per scheduler: DFMA
// 8.8 cycles dependent / 2.1 issue, SHFL 26 / 4.5 and one per cycle for the whole SM, F2F ~10 issue, a barrier of 16 warps
// ~50): so the owners are the first n threads (few warps convert and integrate, the others only help with the pairs), and
// nothing on the per-evaluation path is reduced by shuffles.
//
// LIST PATH (n <= 64 L and the table fits: the sparse chains of a planetesimal disc).  The n^2 examinations are done in
// FP32 against a threshold widened by more than the FP32 rounding AND by the skin BC_SKIN rc, L lanes per body; the k-th
// hit of body i goes to entry (k + 1) npad + i of the table S.part (k from a prefix sum over the body's L lanes: one
// barrier, no block-wide compaction).  The table is then KEPT: the owners check that no body has moved, after the rigid
// motion that takes the central body back to where it was (a rigid motion keeps every distance), by more than half the
// skin; if so no pair outside the table can have come inside rc_ij and the n^2 pass is skipped.  While they check, the
// warps that own nothing already evaluate the table (bc_pairs: exact FP64 test and both changeover weights of every
// listed ordered pair, zero where it is outside rc_ij; row 0: the star); if the check fails their work is thrown
// away and a new table is made.  At 70 % of the skin the table is used once more and dropped; a round starts with a new
// one (the state has jumped), and trial steps so long that a table never survives to its first check (lst.span_fail:
// differential rotation moves the members of a group against each other by more than the skin) make a new one every time
// without trying.  The owner adds up its own column of the table, top to bottom.
// Dense or very large groups keep the direct loop: the lanes of a body evaluate their own hits and reduce by shuffles.
// One thread copies *watch (the master's round number) into S.bc[buf] before the first barrier of this evaluation; the
// value every thread finds there afterwards is returned.
template <int MAXN, int THREADS>
__device__ __forceinline__ int bc_rhs2(BcSmem<MAXN, THREADS> &S, const BcLane &t, int &buf, double G, double m0,
                                       const double qA[3], const double qB[3], double aA[3], double aB[3],
                                       const volatile int *watch, BcList &lst)
{
    GENGA_BS_RHS_HOOK();
    double(*pA)[MAXN] = S.pos[buf][0];
    double(*pB)[MAXN] = S.pos[buf][1];
    float4 *fA = S.pf[buf][0];
    float4 *fB = S.pf[buf][1];
    if (t.owner) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            pA[c][t.i] = qA[c]; pB[c][t.i] = qB[c];
        }
        const float th = S.thr2[t.i];
        fA[t.i] = make_float4((float)qA[0], (float)qA[1], (float)qA[2], th);
        fB[t.i] = make_float4((float)qB[0], (float)qB[1], (float)qB[2], th);
    }
    if (threadIdx.x == THREADS - 32) S.bc[buf] = *watch;     // a thread that owns nothing: the owners' warp does not wait for this
    __syncthreads();
    const int seen = S.bc[buf];
    const int sb = buf;
    if (threadIdx.x == THREADS - 32) { S.stale[buf ^ 1] = 0; S.kmax[buf ^ 1] = 0; }                  // read last in the evaluation before this one
    buf ^= 1;
    double ax = 0.0, ay = 0.0, az = 0.0, bx = 0.0, by = 0.0, bz = 0.0;
    const int n = t.n, L = t.L, i = t.pi;                         // below, i is the body whose pairs this lane examines
    const bool live = i < n;
    const bool one_chunk = n <= 64 * L;                           // every partner of a lane fits one 64-bit mask (uniform)
    bool summed = false;                                          // the owners already hold their sums
    if (one_chunk) {
        bool listed = false;
        if (lst.valid) {
            // optimistic: the warps that own no body evaluate the listed pairs while the owners check the list; if the
            // check fails (rare), what they wrote is thrown away
            const int ow = (n + 31) & ~31;                        // threads of the owners' warps
            bool still = true;
            if (t.owner) {
                // rigid motion taken out first: the rotation about z that puts the central body back on its old azimuth, then its shift
                const float4 oA = fA[lst.ref], oB = fB[lst.ref], o = S.ref[lst.ref], r = S.ref[t.i], mA = fA[t.i], mB = fB[t.i];
                const float on = o.x * o.x + o.y * o.y;
                const float nA = rsqrtf((oA.x * oA.x + oA.y * oA.y) * on), nB = rsqrtf((oB.x * oB.x + oB.y * oB.y) * on);
                const float cA = (oA.x * o.x + oA.y * o.y) * nA, sA = (oA.x * o.y - oA.y * o.x) * nA;
                const float cB = (oB.x * o.x + oB.y * o.y) * nB, sB = (oB.x * o.y - oB.y * o.x) * nB;
                const float ux = mA.x - oA.x, uy = mA.y - oA.y, wx = mB.x - oB.x, wy = mB.y - oB.y;
                const float rx = r.x - o.x, ry = r.y - o.y, rz = r.z - o.z;
                const float dx = (cA * ux - sA * uy) - rx, dy = (sA * ux + cA * uy) - ry, dz = (mA.z - oA.z) - rz;
                const float ex = (cB * wx - sB * wy) - rx, ey = (sB * wx + cB * wy) - ry, ez = (mB.z - oB.z) - rz;
                const float moved = fmaxf(fmaf(dz, dz, fmaf(dy, dy, dx * dx)), fmaf(ez, ez, fmaf(ey, ey, ex * ex)));
                still = moved < S.skin2;
                if (!(moved < 0.5f * S.skin2)) atomicOr(&S.stale[sb], still ? 2 : 3);     // 2: 70 % of the way: a new list next time
            }
            if (ow < THREADS) bc_pairs(S, pA, pB, G, m0, lst, n, ow);
            __syncthreads();                                      // a plain barrier and a flag: half the price of a voting barrier
            const int st = S.stale[sb];
            listed = !(st & 1);
            if (st) lst.valid = false;                            // this list was used for the last time
            if (!listed && lst.age == 0) lst.span_fail = fmin(lst.span_fail, lst.span);
            ++lst.age;
            if (listed && ow >= THREADS) {                        // no warp to spare: the pairs after the check
                bc_pairs(S, pA, pB, G, m0, lst, n, 0);
                __syncthreads();
            }
        }
        if (!listed) {
            // ---- pretest: bit kk = partner j = s + kk L passed at point A or B.  Four partners per trip, no early exit:
            // their loads and short FP32 chains overlap (one at a time this loop was most of what a new list costs)
            unsigned long long mask = 0ull;
            if (live) {
                const float4 mA = fA[i], mB = fB[i];
                const float ft = mA.w;
                if (t.s == 0) S.ref[i] = mA;
                const int trips = (n - t.s + 4 * L - 1) / (4 * L);    // t.s < L <= n
#pragma unroll 1
                for (int q4 = 0; q4 < trips; ++q4) {
                    unsigned bits = 0u;
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int j = t.s + (4 * q4 + u) * L, jj = min(j, n - 1);
                        const float4 pa = fA[jj], pb = fB[jj];
                        const float dx = pa.x - mA.x, dy = pa.y - mA.y, dz = pa.z - mA.z;
                        const float ex = pb.x - mB.x, ey = pb.y - mB.y, ez = pb.z - mB.z;
                        const float d2 = fminf(fmaf(dz, dz, fmaf(dy, dy, dx * dx)), fmaf(ez, ez, fmaf(ey, ey, ex * ex)));
                        bits |= (d2 < fmaxf(ft, pa.w) && j != i && j < n) ? 1u << u : 0u;
                    }
                    mask |= (unsigned long long)bits << (4 * q4);
                }
            }
            // ---- the k-th hit of body i goes to entry (k + 1) npad + i: k from a prefix sum over the body's L lanes only, so
            // the table is complete after ONE barrier (no block-wide compaction)
            const int lane = threadIdx.x & 31;
            const int cnt = __popcll(mask);
            int pre = cnt;
            for (int o = 1; o < L; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, pre, o, L); if (t.s >= o) pre += v; }
            const int cseg = __shfl_sync(0xffffffffu, pre, L - 1, L);           // the body's partners
            const int wmax = __reduce_max_sync(0xffffffffu, cseg);
            if (lane == 0 && wmax > 0) atomicMax(&S.kmax[sb], wmax);
            const int npad = lst.npad;
            if (live) {
                if (t.s == 0) S.cnt[i] = cseg;
                int slot = (pre - cnt + 1) * npad + i;
                for (unsigned long long mm = mask; mm && slot < BC_MAXP; mm &= mm - 1, slot += npad) S.part[slot] = t.s + (__ffsll((long long)mm) - 1) * L;
            }
            __syncthreads();
            const int kmax = S.kmax[sb];
            listed = (kmax + 1) * npad <= BC_MAXP;
            lst.valid = listed && S.skin2 > 0.f && lst.span < lst.span_fail;
            lst.age = 0;
            lst.rows = kmax + 1;
            if (listed) {
                bc_pairs(S, pA, pB, G, m0, lst, n, 0);
                __syncthreads();
            } else if (live) {
                // ---- dense group: the lanes evaluate their own hits
                const double xA = pA[0][i], yA = pA[1][i], zA = pA[2][i], xB = pB[0][i], yB = pB[1][i], zB = pB[2][i];
                const double my_rc = S.rc[i], my_irc = S.irc[i];
                while (mask) {
                    const int j = t.s + (__ffsll((long long)mask) - 1) * L;
                    mask &= mask - 1;
                    double rcj = S.rc[j];
                    double rcij = fmax(my_rc, rcj), rc2 = rcij * rcij;
                    double dx = pA[0][j] - xA, dy = pA[1][j] - yA, dz = pA[2][j] - zA;
                    double ex = pB[0][j] - xB, ey = pB[1][j] - yB, ez = pB[2][j] - zB;
                    double dA = dx * dx + dy * dy + dz * dz, dB = ex * ex + ey * ey + ez * ez;
                    const bool inA = dA < rc2, inB = dB < rc2;
                    if (inA || inB) {
                        const double ir = my_rc >= rcj ? my_irc : S.irc[j], gmj = G * S.m[j];
                        double scA = direct_scale_nb(inA ? dA : rc2, rcij, ir, gmj);
                        double scB = direct_scale_nb(inB ? dB : rc2, rcij, ir, gmj);
                        scA = inA ? scA : 0.0; scB = inB ? scB : 0.0;
                        ax += scA * dx; ay += scA * dy; az += scA * dz;
                        bx += scB * ex; by += scB * ey; bz += scB * ez;
                    }
                }
            }
        }
        if (listed) {
            // ---- the owner: the star, then its own range in list order; four entries per trip (their loads in flight
            // together), then one by one: as few instructions as possible, the owners' warp is alone on this stretch
            if (t.owner) {
                const int row = 6 * lst.npad;
                const double *e = S.pres[t.i];
                int left = S.cnt[t.i];
                double2 v0 = *reinterpret_cast<const double2 *>(e), v1 = *reinterpret_cast<const double2 *>(e + 2), v2 = *reinterpret_cast<const double2 *>(e + 4);
                ax = v0.x; ay = v0.y; az = v1.x; bx = v1.y; by = v2.x; bz = v2.y;
                e += row;
#pragma unroll 1
                for (; left >= 4; left -= 4, e += 4 * row) {
                    const double *f = e + row, *g = f + row, *h = g + row;
                    const double2 a0 = *reinterpret_cast<const double2 *>(e), a1 = *reinterpret_cast<const double2 *>(e + 2), a2 = *reinterpret_cast<const double2 *>(e + 4);
                    const double2 b0 = *reinterpret_cast<const double2 *>(f), b1 = *reinterpret_cast<const double2 *>(f + 2), b2 = *reinterpret_cast<const double2 *>(f + 4);
                    const double2 c0 = *reinterpret_cast<const double2 *>(g), c1 = *reinterpret_cast<const double2 *>(g + 2), c2 = *reinterpret_cast<const double2 *>(g + 4);
                    const double2 d0 = *reinterpret_cast<const double2 *>(h), d1 = *reinterpret_cast<const double2 *>(h + 2), d2 = *reinterpret_cast<const double2 *>(h + 4);
                    ax += (a0.x + b0.x) + (c0.x + d0.x); ay += (a0.y + b0.y) + (c0.y + d0.y); az += (a1.x + b1.x) + (c1.x + d1.x);
                    bx += (a1.y + b1.y) + (c1.y + d1.y); by += (a2.x + b2.x) + (c2.x + d2.x); bz += (a2.y + b2.y) + (c2.y + d2.y);
                }
#pragma unroll 1
                for (; left > 0; --left, e += row) {
                    v0 = *reinterpret_cast<const double2 *>(e); v1 = *reinterpret_cast<const double2 *>(e + 2); v2 = *reinterpret_cast<const double2 *>(e + 4);
                    ax += v0.x; ay += v0.y; az += v1.x; bx += v1.y; by += v2.x; bz += v2.y;
                }
            }
            summed = true;
        }
    } else if (live) {
        const float4 mA = fA[i], mB = fB[i];
        const float ft = mA.w;
        const double xA = pA[0][i], yA = pA[1][i], zA = pA[2][i], xB = pB[0][i], yB = pB[1][i], zB = pB[2][i];
        const double my_rc = S.rc[i], my_irc = S.irc[i];
        for (int j0 = t.s; j0 < n; j0 += 32 * L) {
            unsigned mask = 0u;
#pragma unroll 4
            for (int kk = 0; kk < 32; ++kk) {
                int j = j0 + kk * L;
                if (j >= n) break;
                const float4 pa = fA[j], pb = fB[j];
                float dx = pa.x - mA.x, dy = pa.y - mA.y, dz = pa.z - mA.z;
                float ex = pb.x - mB.x, ey = pb.y - mB.y, ez = pb.z - mB.z;
                float d2 = fminf(fmaf(dz, dz, fmaf(dy, dy, dx * dx)), fmaf(ez, ez, fmaf(ey, ey, ex * ex)));
                bool in = d2 < fmaxf(ft, pa.w) && j != i;
                mask |= (in ? 1u : 0u) << kk;
            }
            // pairs that passed: exact test, then both changeover weights in one straight-line block (no branch inside,
            // so the two dependent chains overlap and the lanes of a warp do not split)
            while (mask) {
                int j = j0 + (__ffs(mask) - 1) * L;
                mask &= mask - 1;
                double rcj = S.rc[j];
                double rcij = fmax(my_rc, rcj), rc2 = rcij * rcij;
                double dx = pA[0][j] - xA, dy = pA[1][j] - yA, dz = pA[2][j] - zA;
                double ex = pB[0][j] - xB, ey = pB[1][j] - yB, ez = pB[2][j] - zB;
                double dA = dx * dx + dy * dy + dz * dz, dB = ex * ex + ey * ey + ez * ez;
                const bool inA = dA < rc2, inB = dB < rc2;
                if (inA || inB) {
                    const double ir = my_rc >= rcj ? my_irc : S.irc[j], gmj = G * S.m[j];
                    double scA = direct_scale_nb(inA ? dA : rc2, rcij, ir, gmj);
                    double scB = direct_scale_nb(inB ? dB : rc2, rcij, ir, gmj);
                    scA = inA ? scA : 0.0; scB = inB ? scB : 0.0;
                    ax += scA * dx; ay += scA * dy; az += scA * dz;
                    bx += scB * ex; by += scB * ey; bz += scB * ez;
                }
            }
        }
    }
    if (!summed) {
        // ---- direct loops: lane 0 of the body adds the star; the L partial sums are reduced by an xor-butterfly (fixed
        // order) and handed to the owner thread through S.pres
        if (live) {
            const double xA = pA[0][i], yA = pA[1][i], zA = pA[2][i], xB = pB[0][i], yB = pB[1][i], zB = pB[2][i];
            double rA = xA * xA + yA * yA + zA * zA, rB = xB * xB + yB * yB + zB * zB;
            double sA = -G * m0 * rinv3_fast(rA), sB = -G * m0 * rinv3_fast(rB);
            sA = t.s == 0 ? sA : 0.0; sB = t.s == 0 ? sB : 0.0;
            ax += sA * xA; ay += sA * yA; az += sA * zA;
            bx += sB * xB; by += sB * yB; bz += sB * zB;
        }
        for (int o = L >> 1; o > 0; o >>= 1) {
            ax += __shfl_xor_sync(0xffffffffu, ax, o); ay += __shfl_xor_sync(0xffffffffu, ay, o); az += __shfl_xor_sync(0xffffffffu, az, o);
            bx += __shfl_xor_sync(0xffffffffu, bx, o); by += __shfl_xor_sync(0xffffffffu, by, o); bz += __shfl_xor_sync(0xffffffffu, bz, o);
        }
        if (live && t.s == 0) {
            double *o = S.pres[i];
            o[0] = ax; o[1] = ay; o[2] = az; o[3] = bx; o[4] = by; o[5] = bz;
        }
        __syncthreads();
        if (t.owner) {
            const double *o = S.pres[t.i];
            ax = o[0]; ay = o[1]; az = o[2]; bx = o[3]; by = o[4]; bz = o[5];
        }
    }
    aA[0] = ax; aA[1] = ay; aA[2] = az;
    aB[0] = bx; aB[1] = by; aB[2] = bz;
    return seen;
}

// Orders this thread's accesses to the shared memory of the cluster's CTAs (the round record, the column results, the
// flags): cluster scope is enough, and far cheaper than the device-wide fence with its L1 invalidation.
__device__ __forceinline__ void bc_fence() { asm volatile("fence.acq_rel.cluster;" ::: "memory"); }
// Polling a flag another CTA of the cluster sets after it has fenced its data: an acquire load (measured ~30 cycles; a
// fence after a plain load ~290, it is a device-wide MEMBAR with an L1 invalidation whatever scope is asked for).
__device__ __forceinline__ int bc_ld_acquire(const volatile int *flag)
{
    int v;
    const unsigned a = (unsigned)__cvta_generic_to_shared(const_cast<const int *>(flag));
    asm volatile("ld.acquire.cluster.shared::cta.b32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
    return v;
}

template <int MAXN, int THREADS>
__device__ __forceinline__ double bc_block_max(BcSmem<MAXN, THREADS> &S, double v)
{
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    __syncthreads();
    if ((threadIdx.x & 31) == 0) S.red[threadIdx.x >> 5] = v;
    __syncthreads();
    double r = S.red[0];
#pragma unroll
    for (int w = 1; w < THREADS / 32; ++w) r = fmax(r, S.red[w]);
    return r;
}

// thread 0 spins until *flag != old; every thread gets the value it saw
template <int MAXN, int THREADS>
__device__ __forceinline__ int bc_wait_change(BcSmem<MAXN, THREADS> &S, const volatile int *flag, int old)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        int v;
        while ((v = bc_ld_acquire(flag)) == old) __nanosleep(20);      // what the writer stored before the flag is visible to this thread, and after the barrier to the block
        S.bc[0] = v;
    }
    __syncthreads();
    return S.bc[0];
}

// Checker: row k of the Aitken-Neville tableau in (H/n_k)^2 from the column results T[0..k][0] of this level:
// eight lanes per body, six of them take one component each.  Returns the largest scaled squared correction
// max_i max(|dq_i|^2 / |q_i|^2, |dV_i|^2 / |V_i|^2) of T[k][k] - T[k][k-1] (the same in every thread) and leaves
// T[k][k] in S.diag.
template <int MAXN, int THREADS>
__device__ __forceinline__ double bc_check_row(BcSmem<MAXN, THREADS> &S, const int n, const int k)
{
    double e = 0.0;
    for (int i8 = threadIdx.x >> 3; i8 < ((n + 3) & ~3); i8 += THREADS / 8) {
        const int c = threadIdx.x & 7;
        double d2 = 0.0;
        if (c < 6 && i8 < n) {
            double T[BS_KMAX];
#pragma unroll
            for (int r = 0; r < BS_KMAX; ++r) T[r] = r <= k ? S.tab[r][c][i8] : 0.0;
            double last = 0.0;
            // column by column, rows from the bottom up, in place (bs_warp.cuh bw_neville): T[r] <- T[r][j]
#pragma unroll
            for (int j = 1; j < BS_KMAX; ++j) {
                if (j <= k) {
#pragma unroll
                    for (int r = BS_KMAX - 1; r >= j; --r) {
                        if (r <= k) {
                            const double nxt = T[r] + (T[r] - T[r - 1]) * c_bs_iden.v[r][j];
                            if (r == k && j == k) last = nxt - T[r];
                            T[r] = nxt;
                        }
                    }
                }
            }
            double tk = T[0];
#pragma unroll
            for (int r = 1; r < BS_KMAX; ++r) tk = r == k ? T[r] : tk;
            S.diag[c][i8] = tk;
            d2 = last * last;
        }
        const int base = (threadIdx.x & 31) & ~7;
        const double isq = i8 < n ? S.isq[i8] : 0.0, isv = i8 < n ? S.isv[i8] : 0.0;
        const double dq = __shfl_sync(0xffffffffu, d2, base) + __shfl_sync(0xffffffffu, d2, base + 1) + __shfl_sync(0xffffffffu, d2, base + 2);
        const double dv = __shfl_sync(0xffffffffu, d2, base + 3) + __shfl_sync(0xffffffffu, d2, base + 4) + __shfl_sync(0xffffffffu, d2, base + 5);
        e = fmax(e, fmax(dq * isq, dv * isv));
    }
    return bc_block_max(S, e);
}

// The same for groups of at most THREADS / 8 bodies (one tableau entry per thread), row after row: the thread keeps the
// previous row T[k-1][0..k-1] of its entry in prow, so row k costs k steps of the recurrence instead of the whole
// triangle, with the same operands in the same order (the result is bit for bit the one of bc_check_row).
template <int MAXN, int THREADS>
__device__ __forceinline__ double bc_check_row_inc(BcSmem<MAXN, THREADS> &S, const int n, const int k, double (&prow)[BS_KMAX])
{
    const int i8 = threadIdx.x >> 3, c = threadIdx.x & 7;
    double d2 = 0.0;
    if (c < 6 && i8 < n) {
        if (k == 1) prow[0] = S.tab[0][c][i8];
        double cur = S.tab[k][c][i8], prev = prow[0], diff = 0.0;
        prow[0] = cur;
#pragma unroll
        for (int j = 1; j < BS_KMAX; ++j) {
            if (j <= k) {
                const double tmp = prow[j];
                const double nxt = cur + (cur - prev) * c_bs_iden.v[k][j];
                diff = nxt - cur;
                cur = nxt;
                prow[j] = cur;
                prev = tmp;
            }
        }
        S.diag[c][i8] = cur;
        d2 = diff * diff;
    }
    const int base = (threadIdx.x & 31) & ~7;
    const double isq = i8 < n ? S.isq[i8] : 0.0, isv = i8 < n ? S.isv[i8] : 0.0;
    const double dq = __shfl_sync(0xffffffffu, d2, base) + __shfl_sync(0xffffffffu, d2, base + 1) + __shfl_sync(0xffffffffu, d2, base + 2);
    const double dv = __shfl_sync(0xffffffffu, d2, base + 3) + __shfl_sync(0xffffffffu, d2, base + 4) + __shfl_sync(0xffffffffu, d2, base + 5);
    return bc_block_max(S, fmax(dq * isq, dv * isv));
}

// Master: does a pair of the group collide in the step just accepted (L328: the Hermite minimum of Eq. 10-12 over the
// step against (R_a + R_b)^2)?  Old state S.Y, new state SW->diag.  The same answer in every thread.
template <int MAXN, int THREADS>
__device__ __noinline__ bool bc_any_collision(BcSmem<MAXN, THREADS> &S, const BcSmem<MAXN, THREADS> *SW, const int n, const double H)
{
    int hit = 0;
    for (int a = threadIdx.x; a < n && !hit; a += THREADS) {
        if (S.R[a] < 0.0) continue;
        double qa0[3], va0[3], qa1[3], va1[3];
        for (int c = 0; c < 3; ++c) { qa0[c] = S.Y[c][a]; va0[c] = S.Y[3 + c][a]; qa1[c] = SW->diag[c][a]; va1[c] = SW->diag[3 + c][a]; }
        for (int b = a + 1; b < n; ++b) {
            if (S.R[b] < 0.0) continue;
            double P0 = 0.0, Pd0 = 0.0, P1 = 0.0, Pd1 = 0.0;
            for (int c = 0; c < 3; ++c) {
                const double d0 = S.Y[c][b] - qa0[c], w0 = S.Y[3 + c][b] - va0[c];
                const double d1 = SW->diag[c][b] - qa1[c], w1 = SW->diag[3 + c][b] - va1[c];
                P0 += d0 * d0; Pd0 += 2.0 * d0 * w0; P1 += d1 * d1; Pd1 += 2.0 * d1 * w1;
            }
            if (pair_collides(P0, P1, Pd0, Pd1, H, S.R[a] + S.R[b])) { hit = 1; break; }
        }
    }
    return __syncthreads_or(hit) != 0;
}

// One group, integrated over h by the whole cluster of 8 LV CTAs (rank = this CTA's rank in it: level rank / 8,
// column rank % 8).  On entry S.Y, S.m, S.rc, S.irc of EVERY CTA hold the group; seq = the last round number used (the
// same in every CTA; 0 and the protocol words of S zero at kernel start), updated on return.  On return S.Y of the
// master (rank 0) holds the result.  Returns false on step-size underflow (uniform over the cluster).  nsteps (master
// only): [0] accepted steps, [1] rejected attempts as the sequential rule counts them.
// Returns 0: step size underflow, 1: done, 2 (coll != 0): a pair of the group collides in an accepted step; the group is
// abandoned (k_bs_generic integrates it again and merges the pair).
template <int MAXN, int THREADS, int LV>
__device__ __forceinline__ int bc_integrate(BcSmem<MAXN, THREADS> &S, const int rank, const BcLane &t, double G, double m0,
                                            double h, double eps, int *nsteps, int &seq, const int coll)
{
    using Smem = BcSmem<MAXN, THREADS>;
    cg::cluster_group cluster = cg::this_cluster();
    constexpr int NCTA = BS_KMAX * LV;
    const int lev = rank / BS_KMAX, col = rank % BS_KMAX;
    const bool master = rank == 0, checker = col == 0;
    Smem *SC = cluster.map_shared_rank(&S, lev * BS_KMAX);       // my level's checker
    Smem *S0 = cluster.map_shared_rank(&S, 0);                   // the master
    const int i = t.i, n = t.n, tid = threadIdx.x;
    const double eps2 = eps * eps;
    int buf = 0;
    __syncthreads();
    {
        // FP32 pretest thresholds: positions stay within Q = 2 max_i(|q_i| + |h| |V_i|) (max norms) of
        // the origin during the step, so rounding them to FP32 moves a separation by < 2^-22 Q and
        // the FP32 evaluation of its square adds < 2^-21 relative; thr = (rc + 2^-20 Q)^2 (1 + 2^-18).
        double qm = 0.0;
        if (t.owner) {
            qm = fmax(fmax(fabs(S.Y[0][i]), fabs(S.Y[1][i])), fabs(S.Y[2][i])) +
                 fabs(h) * fmax(fmax(fabs(S.Y[3][i]), fabs(S.Y[4][i])), fabs(S.Y[5][i]));
        }
        const double Q = 2.0 * bc_block_max(S, qm);
        // List path of bc_rhs2 (n <= 32 L): the pretest reaches out to (1 + BC_SKIN) rc, and the list is kept while every
        // body stays within skin = BC_SKIN min_i rc_i / 2 of where it was, in the frame of the central body, when the list was made
        // (less 2^-19 Q for the FP32 roundings of that difference): a pair left out cannot have come inside rc_ij.
        const bool wide = n <= 64 * t.L;
        const double rcmin = -bc_block_max(S, t.owner ? -S.rc[i] : -1.0e300);
        if (t.owner) {
            double w = S.rc[i] * (wide ? 1.0 + BC_SKIN : 1.0) + 0x1.0p-20 * Q;
            S.thr2[i] = __double2float_ru(w * w * (1.0 + 0x1.0p-18));
        }
        if (tid == 0) {
            const double sk = 0.5 * BC_SKIN * rcmin - 0x1.0p-19 * Q;
            S.skin2 = wide && sk > 0.0 ? __double2float_rd(sk * sk * (1.0 - 0x1.0p-18)) : 0.f;
            S.stale[0] = 0; S.stale[1] = 0; S.kmax[0] = 0; S.kmax[1] = 0;
            // the body nearest the centre of the group: differential rotation moves the others least against its frame
            double cx = 0.0, cy = 0.0, cz = 0.0;
            for (int b = 0; b < n; ++b) { cx += S.Y[0][b]; cy += S.Y[1][b]; cz += S.Y[2][b]; }
            cx /= n; cy /= n; cz /= n;
            int best = 0;
            double bd = 1.0e300;
            for (int b = 0; b < n; ++b) {
                const double dx = S.Y[0][b] - cx, dy = S.Y[1][b] - cy, dz = S.Y[2][b] - cz, dd = dx * dx + dy * dy + dz * dz;
                if (dd < bd) { bd = dd; best = b; }
            }
            S.refbody = best;
        }
        __syncthreads();
    }
    BcList lst;
    lst.rows = 1; lst.npad = n | 1; lst.magic = 0xffffffffu / (unsigned)(n | 1) + 1u; lst.valid = false;
    lst.age = 0; lst.span = 0.0; lst.span_fail = 1.0e300; lst.ref = S.refbody;
    // ---- master: the step-size control of the sequential algorithm; everybody: rounds as they are published
    double done = 0.0, H = h;
    bool last = true;                             // the first trial step is the whole interval
    if (master && tid < NCTA) {                   // first round of this group: the state is already in every CTA
        Smem *R = cluster.map_shared_rank(&S, tid);
        R->seq_begin = seq + 1; R->rec_H = H; R->rec_state = 0;
        bc_fence();
        R->seq_end = seq + 1;
    }
    int ok = 1;
#ifdef GENGA_BC_PROF
    long long pf_t = clock64(), pf_acc[6] = {0, 0, 0, 0, 0, 0};   // record, rhs, wait, check, publish, calls
#define BC_PROF(k) { const long long now_ = clock64(); pf_acc[k] += now_ - pf_t; pf_t = now_; }
#else
#define BC_PROF(k)
#endif
    while (true) {
        // ---- the newest record (sequence lock: the master may be rewriting it)
        int e, state;
        double Hr;
        bool consistent;
        double q[3] = {1.0, 0.0, 0.0}, V[3] = {0.0, 1.0, 0.0};
        do {
            e = bc_wait_change(S, &S.seq_end, seq);
            Hr = S.rec_H; state = S.rec_state;
            if (t.owner) {
#pragma unroll
                for (int c = 0; c < 3; ++c) { q[c] = S.Y[c][i]; V[c] = S.Y[3 + c][i]; }
            }
            if (checker && state == 0) {
                for (int b = tid; b < n; b += THREADS) {
                    const double x = S.Y[0][b], y = S.Y[1][b], z = S.Y[2][b], vx = S.Y[3][b], vy = S.Y[4][b], vz = S.Y[5][b];
                    S.isq[b] = rcp_fast(x * x + y * y + z * z);
                    S.isv[b] = rcp_fast(vx * vx + vy * vy + vz * vz);
                }
            }
            __syncthreads();                      // every thread has read its part of the record
            if (tid == 0) { bc_fence(); S.ok = S.seq_begin == e ? 1 : 0; }
            __syncthreads();
            consistent = S.ok != 0;
        } while (!consistent);
        seq = e;
        lst.valid = false;                        // the state has jumped: the old list fails its check more often than not
        BC_PROF(0)
        if (state != 0) { ok = state == 1 ? 1 : state == 3 ? 2 : 0; break; }
        const double Hl = ldexp(Hr, -lev);
        const bool under = lev > 0 && fabs(Hl) < BS_HMIN * fabs(h);
        bool dropped = false;
        if (!under) {
            // ---- force at the starting state, then my column: Gragg's modified midpoint rule with 2 (col + 1) substeps,
            // two per evaluation (bc_rhs2): q_{k+1} = q_{k-1} + 2 eta V_k does not need a(q_k)
            double acc0[3], dummy[3];
            dropped = bc_rhs2(S, t, buf, G, m0, q, q, acc0, dummy, &S.seq_end, lst) != seq;
            const double eta = Hl / (2 * (col + 1));
            lst.span = fabs(2.0 * eta);
            double qa[3] = {1.0, 0.0, 0.0}, Va[3] = {0.0, 0.0, 0.0}, qb[3] = {1.0, 0.0, 0.0}, Vb[3] = {0.0, 0.0, 0.0};
            if (t.owner) {                        // the other warps only help with the pairs (bc_rhs2)
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    qa[c] = q[c]; Va[c] = V[c];
                    qb[c] = q[c] + eta * V[c]; Vb[c] = V[c] + eta * acc0[c];
                }
            }
#pragma unroll 1
            for (int it = 0; it <= col && !dropped; ++it) {
                double qc[3] = {1.0, 0.0, 0.0}, A[3], C[3];
                if (t.owner) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) qc[c] = qa[c] + 2.0 * eta * Vb[c];
                }
                dropped = bc_rhs2(S, t, buf, G, m0, qb, qc, A, C, &S.seq_end, lst) != seq;    // a newer round: drop this one
                if (t.owner) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        double vc = Va[c] + 2.0 * eta * A[c];
                        if (it == col && !dropped) {
                            SC->tab[col][c][i] = 0.5 * (qc[c] + qb[c] + eta * vc);
                            SC->tab[col][3 + c][i] = 0.5 * (vc + Vb[c] + eta * C[c]);
                        }
                        double qd = qb[c] + 2.0 * eta * vc, vd = Vb[c] + 2.0 * eta * C[c];
                        qa[c] = qc[c]; Va[c] = vc; qb[c] = qd; Vb[c] = vd;
                    }
                }
            }
            if (!dropped) {
                __syncthreads();                  // the owners' column results are on their way to the checker
                if (tid == 0) { bc_fence(); SC->ready[col] = seq; }
            }
        }
        BC_PROF(1)
        if (!checker) continue;
        // ---- checker of this level: rows 1.. as their columns arrive; first row whose error passes
        int code = under ? 0 : 1;                 // 0 underflow, 1 rejected, 2 + k passed at row k
        double prow[BS_KMAX] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        if (!under && !dropped) {
            for (int k = 1; k < BS_KMAX; ++k) {
                // wait for column k of this round (or for a newer round: checkers of the levels behind the first)
                __syncthreads();
                if (tid == 0) {
                    int a;
                    while ((a = bc_ld_acquire(&S.ready[k])) != seq && S.seq_end == seq) __nanosleep(20);
                    S.bc[0] = a == seq ? 1 : 0;
                }
                __syncthreads();
                if (S.bc[0] == 0) { dropped = true; break; }
                BC_PROF(2)
                const double err = n <= THREADS / 8 ? bc_check_row_inc(S, n, k, prow) : bc_check_row(S, n, k);
                BC_PROF(3)
                if (err <= eps2) { code = 2 + k; break; }
            }
        }
        if (dropped) continue;
        if (!master) {                            // report; T[k][k] stays in S.diag for the master
            __syncthreads();
            if (tid == 0) { bc_fence(); S0->lev_result[lev] = (seq << 8) | code; }
            continue;
        }
        // ---- master: the first level, in the order H, H/2, .., that passed
        int winner = -1, wrow = 0;
        bool fail = false;
        if (code >= 2) { winner = 0; wrow = code - 2; }
        else {
#pragma unroll 1
            for (int l = 1; l < LV; ++l) {
                __syncthreads();
                if (tid == 0) {
                    int v;
                    while (((v = bc_ld_acquire(&S.lev_result[l])) >> 8) != seq) __nanosleep(20);
                    S.bc[0] = v & 255;
                }
                __syncthreads();
                const int cl = S.bc[0];
                if (cl >= 2) { winner = l; wrow = cl - 2; break; }
                if (cl == 0) { fail = true; break; }
            }
        }
        // a record will be published whatever the outcome: its sequence number goes out first (a reader that finds
        // seq_begin != seq_end knows the record is being rewritten), now, so that its fence overlaps the work below
        const int ns = seq + 1;
        __syncthreads();
        if (tid < NCTA) {
            cluster.map_shared_rank(&S, tid)->seq_begin = ns;
            bc_fence();
        }
        int next_state = 0;
        if (fail) next_state = 2;
        else if (winner >= 0 && coll && bc_any_collision(S, cluster.map_shared_rank(&S, winner * BS_KMAX), n, ldexp(Hr, -winner))) next_state = 3;
        else if (winner >= 0) {
            // the accepted state T[k][k] of the winning level becomes the master's Y (pushed to the others below)
            const Smem *SW = cluster.map_shared_rank(&S, winner * BS_KMAX);
            for (int k = tid; k < n; k += THREADS) {
#pragma unroll
                for (int c = 0; c < 6; ++c) S.Y[c][k] = SW->diag[c][k];
            }
            const double Hw = ldexp(Hr, -winner);
            done += Hw; H = Hw;
            if (nsteps) { ++nsteps[0]; nsteps[1] += winner; }
            if (wrow <= 4) H *= 1.5;
            if (winner > 0) last = false;
            if (last) next_state = 1;
        } else {
            if (nsteps) nsteps[1] += LV;
            H = ldexp(Hr, -LV); last = false;
            if (fabs(H) < BS_HMIN * fabs(h)) next_state = 2;
        }
        if (next_state == 0) {
            const double rem = h - done;
            if (fabs(rem) <= 8.0 * 2.220446049250313e-16 * fabs(h)) next_state = 1;     // a remainder of a few ulp of h: done
            else if (fabs(H) >= fabs(rem)) { H = rem; last = true; }
        }
        // ---- publish the next record (and the new state) to every CTA of the cluster, then the sequence number again.
        // Lane r of the first warp writes the words of CTA r; the state goes out in 16-byte stores (two bodies of one
        // component), spread over the block: what a store to another CTA's shared memory costs is the packet, not its size
        // (8-byte stores: 2.9 k cycles for 30 bodies, measured).
        __syncthreads();                          // seq_begin is out (fenced), the master's Y is complete
        if (winner >= 0 && next_state == 0) {
            const int np2 = (n + 1) >> 1;         // pairs of bodies (Y rows are MAXN long, MAXN even: the odd one out copies a spare)
            for (int idx = tid; idx < np2 * NCTA; idx += THREADS) {
                const int r = idx % NCTA, kp = idx / NCTA;
                if (r == 0) continue;
                Smem *R = cluster.map_shared_rank(&S, r);
#pragma unroll
                for (int c = 0; c < 6; ++c) *reinterpret_cast<double2 *>(&R->Y[c][2 * kp]) = *reinterpret_cast<const double2 *>(&S.Y[c][2 * kp]);
            }
        }
        if (tid < NCTA) {
            Smem *R = cluster.map_shared_rank(&S, tid);
            R->rec_H = H; R->rec_state = next_state;
        }
        __syncthreads();
        if (tid < NCTA) { bc_fence(); cluster.map_shared_rank(&S, tid)->seq_end = ns; }
        BC_PROF(4)
    }
#ifdef GENGA_BC_PROF
    if (master && tid == 0 && nsteps) { for (int k = 0; k < 5; ++k) nsteps[2 + k] = (int)(pf_acc[k] >> 4); }
#endif
    return ok;
}

}  // namespace genga
