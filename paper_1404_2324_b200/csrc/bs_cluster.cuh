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
// Inside a CTA, body i owns L adjacent lanes (a power of two, at most a warp); lane s of the segment takes partners
// j = s, s+L, ...; the segment sum is an xor-butterfly (fixed order); lane 0 of the segment ("owner") carries the
// body's midpoint state in registers.  Positions are exchanged through a double-buffered shared array: one
// __syncthreads per force evaluation.
#pragma once
#include <cooperative_groups.h>
#include <cstdio>

#include "bs.cuh"

namespace genga {

namespace cg = cooperative_groups;

constexpr int BC_MAXP = 768;         // ordered close pairs the list path of bc_rhs2 takes (sparse groups: a few per body)

template <int MAXN, int THREADS>
struct BcSmem {
    double pos[2][2][3][MAXN];      // [buffer][point A / B][component][body]
    float4 pf[2][2][MAXN];          // positions rounded to FP32 for the conservative pretest, .w = thr2: one LDS.128 per partner
    double isq[MAXN], isv[MAXN];    // checker: 1 / |q|^2, 1 / |V|^2 of the round's starting state (error norm)
    float thr2[MAXN];               // (rc_i + margin)^2 rounded up
    double m[MAXN], rc[MAXN], irc[MAXN];
    double R[MAXN];                 // physical radii (collision test; < 0: none)
    double Y[6][MAXN];              // state the current round starts from (pushed by the master)
    double tab[BS_KMAX][6][MAXN];   // checker: column results T[k][0] of its level
    double diag[6][MAXN];           // checker: T[k][k] of the row tested last
    double red[THREADS / 32];
    // ---- close pairs of the current evaluation (bc_rhs2, list path)
    int2 plist[BC_MAXP];            // ordered pairs (i, j) that passed the FP32 pretest at either point, body by body
    double pres[BC_MAXP][6];        // their geometric factors times the separation at the two points (without G m_j)
    int wtot[THREADS / 32];         // pairs found by each warp
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
    int n, L, i, s;
    bool owner;
};

template <int THREADS>
__device__ __forceinline__ BcLane bc_lanes(int n)
{
    int P = 2;
    while (P < n) P <<= 1;              // bodies, rounded up to a power of two
    BcLane t;
    t.n = n; t.L = min(8, THREADS / P);  // lanes per body: they only pretest and gather (bc_rhs2)
    t.i = threadIdx.x / t.L; t.s = threadIdx.x % t.L;
    t.owner = t.s == 0 && t.i < n;
    return t;
}

// Forces on body t.i at TWO sets of positions (qA, qB of the owners) at once (Eq. 1 L73-74 through Eq. 8
// L104; star fixed at the origin, L314; every pair of the group is examined at every evaluation, L505).
// Two at once because a(q_k) and a(q_{k+1}) of Gragg's rule are independent (bs_warp.cuh): one barrier and
// one segment reduction serve both, and their dependent chains overlap.  The n^2 examinations are done
// first in FP32 against a threshold widened by more than the FP32 rounding, so the test can only err
// towards "inside"; pairs that pass take the exact FP64 test and weight.
//
// What that costs is the exact pass: ~110 FP64 instructions per close pair, and a warp runs them as long as ANY of its
// lanes has a pair left, so with 16 warps on one SM the FP64 pipe was busy ~2.6 k of the 6.5 k cycles of an evaluation
// of a 55-body group, most of it on idle lanes.  LIST PATH (all partners of a lane in one 32-bit mask, at most BC_MAXP
// close ordered pairs: the sparse chains of a planetesimal disc): the lanes only pretest; their hits are compacted into
// one list (block-wide prefix sum, body by body, fixed order), ONE thread per listed pair evaluates the exact weights
// of both points, and body i adds up its own contiguous range of the list: the exact pass shrinks to total / 32 warps.
// Dense or very large groups keep the direct loop.
// Thread 0 copies *watch (the master's round number) into S.bc[buf] before the barrier of this evaluation; the value
// every thread finds there afterwards is returned.
template <int MAXN, int THREADS>
__device__ __forceinline__ int bc_rhs2(BcSmem<MAXN, THREADS> &S, const BcLane &t, int &buf, double G, double m0,
                                       const double qA[3], const double qB[3], double aA[3], double aB[3],
                                       const volatile int *watch)
{
    GENGA_BS_RHS_HOOK();
#ifdef GENGA_BC_PROF
    long long ph_[8]; int phn_ = 0;
#define RHS_PROF() ph_[phn_++] = clock64();
#else
#define RHS_PROF()
#endif
    RHS_PROF()
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
    if (threadIdx.x == 0) S.bc[buf] = *watch;
    __syncthreads();
    const int seen = S.bc[buf];
    RHS_PROF()
    buf ^= 1;
    double ax = 0.0, ay = 0.0, az = 0.0, bx = 0.0, by = 0.0, bz = 0.0;
    const int n = t.n, L = t.L, i = t.i;
    const bool live = i < n;
    const bool one_chunk = n <= 32 * L;                           // every partner of a lane fits one mask (uniform)
    if (one_chunk) {
        // ---- pretest: bit kk = partner j = s + kk L passed at point A or B
        unsigned mask = 0u;
        if (live) {
            const float4 mA = fA[i], mB = fB[i];
            const float ft = mA.w;
#pragma unroll 4
            for (int kk = 0; kk < 32; ++kk) {
                const int j = t.s + kk * L;
                if (j >= n) break;
                const float4 pa = fA[j], pb = fB[j];
                float dx = pa.x - mA.x, dy = pa.y - mA.y, dz = pa.z - mA.z;
                float ex = pb.x - mB.x, ey = pb.y - mB.y, ez = pb.z - mB.z;
                float d2 = fminf(fmaf(dz, dz, fmaf(dy, dy, dx * dx)), fmaf(ez, ez, fmaf(ey, ey, ex * ex)));
                const bool in = d2 < fmaxf(ft, pa.w) && j != i;
                mask |= (in ? 1u : 0u) << kk;
            }
        }
        // ---- block-wide exclusive prefix sum of the hit counts, in thread order (= body by body)
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        const int cnt = __popc(mask);
        int inc = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += v; }
        if (lane == 31) S.wtot[warp] = inc;
        RHS_PROF()
        __syncthreads();
        RHS_PROF()
        int base = 0, total = 0;
#pragma unroll
        for (int w = 0; w < THREADS / 32; ++w) { const int v = S.wtot[w]; base += w < warp ? v : 0; total += v; }
        if (total <= BC_MAXP) {
            int at = base + inc - cnt;
            // my body's range of the list: [start of its first lane, + the counts of its L lanes)
            int cseg = cnt;
            for (int o = L >> 1; o > 0; o >>= 1) cseg += __shfl_xor_sync(0xffffffffu, cseg, o);
            const int start = __shfl_sync(0xffffffffu, at, lane & ~(L - 1));
            for (unsigned mm = mask; mm; mm &= mm - 1) S.plist[at++] = make_int2(i, t.s + (__ffs(mm) - 1) * L);
            __syncthreads();
            RHS_PROF()
            // ---- one thread per listed pair: exact test and both changeover weights, without the partner's mass
            for (int p = threadIdx.x; p < total; p += THREADS) {
                const int2 pr = S.plist[p];
                const double rci = S.rc[pr.x], rcj = S.rc[pr.y];
                const double rcij = fmax(rci, rcj), rc2 = rcij * rcij;
                const double dx = pA[0][pr.y] - pA[0][pr.x], dy = pA[1][pr.y] - pA[1][pr.x], dz = pA[2][pr.y] - pA[2][pr.x];
                const double ex = pB[0][pr.y] - pB[0][pr.x], ey = pB[1][pr.y] - pB[1][pr.x], ez = pB[2][pr.y] - pB[2][pr.x];
                const double dA = dx * dx + dy * dy + dz * dz, dB = ex * ex + ey * ey + ez * ez;
                const bool inA = dA < rc2, inB = dB < rc2;
                const double ir = rci >= rcj ? S.irc[pr.x] : S.irc[pr.y];
                double wA = direct_scale_nb(inA ? dA : rc2, rcij, ir, 1.0);
                double wB = direct_scale_nb(inB ? dB : rc2, rcij, ir, 1.0);
                wA = inA ? wA : 0.0; wB = inB ? wB : 0.0;
                S.pres[p][0] = wA * dx; S.pres[p][1] = wA * dy; S.pres[p][2] = wA * dz;
                S.pres[p][3] = wB * ex; S.pres[p][4] = wB * ey; S.pres[p][5] = wB * ez;
            }
            RHS_PROF()
            __syncthreads();
            RHS_PROF()
            // ---- body i: its own range, lane s takes every L-th entry
            if (live) {
                for (int p = start + t.s; p < start + cseg; p += L) {
                    const double gmj = G * S.m[S.plist[p].y];
                    ax = fma(gmj, S.pres[p][0], ax); ay = fma(gmj, S.pres[p][1], ay); az = fma(gmj, S.pres[p][2], az);
                    bx = fma(gmj, S.pres[p][3], bx); by = fma(gmj, S.pres[p][4], by); bz = fma(gmj, S.pres[p][5], bz);
                }
            }
        } else if (live) {
            // ---- dense group: the lanes evaluate their own hits
            const double xA = pA[0][i], yA = pA[1][i], zA = pA[2][i], xB = pB[0][i], yB = pB[1][i], zB = pB[2][i];
            const double my_rc = S.rc[i], my_irc = S.irc[i];
            while (mask) {
                const int j = t.s + (__ffs(mask) - 1) * L;
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
    if (live) {
        // the star (fixed at the origin): every lane of the body computes it, lane 0 keeps it (no split of the warp)
        const double xA = pA[0][i], yA = pA[1][i], zA = pA[2][i], xB = pB[0][i], yB = pB[1][i], zB = pB[2][i];
        double rA = xA * xA + yA * yA + zA * zA, rB = xB * xB + yB * yB + zB * zB;
        double sA = -G * m0 * rinv3_fast(rA), sB = -G * m0 * rinv3_fast(rB);
        sA = t.s == 0 ? sA : 0.0; sB = t.s == 0 ? sB : 0.0;
        ax += sA * xA; ay += sA * yA; az += sA * zA;
        bx += sB * xB; by += sB * yB; bz += sB * zB;
    }
    for (int o = t.L >> 1; o > 0; o >>= 1) {
        ax += __shfl_xor_sync(0xffffffffu, ax, o); ay += __shfl_xor_sync(0xffffffffu, ay, o); az += __shfl_xor_sync(0xffffffffu, az, o);
        bx += __shfl_xor_sync(0xffffffffu, bx, o); by += __shfl_xor_sync(0xffffffffu, by, o); bz += __shfl_xor_sync(0xffffffffu, bz, o);
    }
    aA[0] = ax; aA[1] = ay; aA[2] = az;
    aB[0] = bx; aB[1] = by; aB[2] = bz;
#ifdef GENGA_BC_PROF
    RHS_PROF()
    if (threadIdx.x == 0 && t.n == 55 && (blockIdx.x & 7) < 2 && seen < 4) {
        printf("rhs n=%d blk=%d seq=%d phases:", t.n, blockIdx.x & 7, seen);
        for (int k = 1; k < phn_; ++k) printf(" %d", (int)(ph_[k] - ph_[k - 1]));
        printf("\n");
    }
#endif
    return seen;
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
        while ((v = *flag) == old) __nanosleep(20);
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
        if (t.owner) {
            double w = S.rc[i] + 0x1.0p-20 * Q;
            S.thr2[i] = __double2float_ru(w * w * (1.0 + 0x1.0p-18));
        }
        __syncthreads();
    }
    // ---- master: the step-size control of the sequential algorithm; everybody: rounds as they are published
    double done = 0.0, H = h;
    bool last = true;                             // the first trial step is the whole interval
    if (master && tid == 0) {                     // first round of this group: the state is already in every CTA
        for (int r = 0; r < NCTA; ++r) {
            Smem *R = cluster.map_shared_rank(&S, r);
            R->seq_begin = seq + 1; R->rec_H = H; R->rec_state = 0;
        }
        __threadfence();
        for (int r = 0; r < NCTA; ++r) cluster.map_shared_rank(&S, r)->seq_end = seq + 1;
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
            __threadfence();
            Hr = S.rec_H; state = S.rec_state;
            if (t.owner) {
#pragma unroll
                for (int c = 0; c < 3; ++c) { q[c] = S.Y[c][i]; V[c] = S.Y[3 + c][i]; }
            }
            if (checker && state == 0) {
                for (int b = tid; b < n; b += THREADS) {
                    const double x = S.Y[0][b], y = S.Y[1][b], z = S.Y[2][b], vx = S.Y[3][b], vy = S.Y[4][b], vz = S.Y[5][b];
                    S.isq[b] = 1.0 / (x * x + y * y + z * z);
                    S.isv[b] = 1.0 / (vx * vx + vy * vy + vz * vz);
                }
            }
            __threadfence();
            consistent = __syncthreads_and(S.seq_begin == e) != 0;
        } while (!consistent);
        seq = e;
        BC_PROF(0)
        if (state != 0) { ok = state == 1 ? 1 : state == 3 ? 2 : 0; break; }
        const double Hl = ldexp(Hr, -lev);
        const bool under = lev > 0 && fabs(Hl) < BS_HMIN * fabs(h);
        bool dropped = false;
        if (!under) {
            // ---- force at the starting state, then my column: Gragg's modified midpoint rule with 2 (col + 1) substeps,
            // two per evaluation (bc_rhs2): q_{k+1} = q_{k-1} + 2 eta V_k does not need a(q_k)
            double acc0[3], dummy[3];
            dropped = bc_rhs2(S, t, buf, G, m0, q, q, acc0, dummy, &S.seq_end) != seq;
            const double eta = Hl / (2 * (col + 1));
            double qa[3], Va[3], qb[3], Vb[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                qa[c] = q[c]; Va[c] = V[c];
                qb[c] = q[c] + eta * V[c]; Vb[c] = V[c] + eta * acc0[c];
            }
#pragma unroll 1
            for (int it = 0; it <= col && !dropped; ++it) {
                double qc[3], A[3], C[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) qc[c] = qa[c] + 2.0 * eta * Vb[c];
                dropped = bc_rhs2(S, t, buf, G, m0, qb, qc, A, C, &S.seq_end) != seq;    // a newer round: drop this one
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    double vc = Va[c] + 2.0 * eta * A[c];
                    if (it == col && t.owner && !dropped) {
                        SC->tab[col][c][i] = 0.5 * (qc[c] + qb[c] + eta * vc);
                        SC->tab[col][3 + c][i] = 0.5 * (vc + Vb[c] + eta * C[c]);
                    }
                    double qd = qb[c] + 2.0 * eta * vc, vd = Vb[c] + 2.0 * eta * C[c];
                    qa[c] = qc[c]; Va[c] = vc; qb[c] = qd; Vb[c] = vd;
                }
            }
            if (!dropped) {
                __threadfence();
                __syncthreads();
                if (tid == 0) SC->ready[col] = seq;
            }
        }
        BC_PROF(1)
        if (!checker) continue;
        // ---- checker of this level: rows 1.. as their columns arrive; first row whose error passes
        int code = under ? 0 : 1;                 // 0 underflow, 1 rejected, 2 + k passed at row k
        if (!under && !dropped) {
            for (int k = 1; k < BS_KMAX; ++k) {
                // wait for column k of this round (or for a newer round: checkers of the levels behind the first)
                __syncthreads();
                if (tid == 0) {
                    int a;
                    while ((a = S.ready[k]) != seq && S.seq_end == seq) __nanosleep(20);
                    S.bc[0] = a == seq ? 1 : 0;
                }
                __syncthreads();
                if (S.bc[0] == 0) { dropped = true; break; }
                __threadfence();
                BC_PROF(2)
                const double err = bc_check_row(S, n, k);
                BC_PROF(3)
                if (err <= eps2) { code = 2 + k; break; }
            }
        }
        if (dropped) continue;
        if (!master) {                            // report; T[k][k] stays in S.diag for the master
            __threadfence();
            __syncthreads();
            if (tid == 0) S0->lev_result[lev] = (seq << 8) | code;
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
                    while (((v = S.lev_result[l]) >> 8) != seq) __nanosleep(20);
                    S.bc[0] = v & 255;
                }
                __syncthreads();
                const int cl = S.bc[0];
                if (cl >= 2) { winner = l; wrow = cl - 2; break; }
                if (cl == 0) { fail = true; break; }
            }
        }
        __threadfence();
        int next_state = 0;
        if (fail) next_state = 2;
        else if (winner >= 0 && coll && bc_any_collision(S, cluster.map_shared_rank(&S, winner * BS_KMAX), n, ldexp(Hr, -winner))) next_state = 3;
        else if (winner >= 0) {
            const Smem *SW = cluster.map_shared_rank(&S, winner * BS_KMAX);
            for (int b = tid; b < 6 * n; b += THREADS) {
                const int c = b / n, k = b - c * n;
                S.Y[c][k] = SW->diag[c][k];
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
        // ---- publish the next record (and the new state) to every CTA of the cluster
        const int ns = seq + 1;
        __syncthreads();
        if (tid == 0) {
            for (int r = 0; r < NCTA; ++r) cluster.map_shared_rank(&S, r)->seq_begin = ns;
            __threadfence();
        }
        __syncthreads();
        if (winner >= 0 && next_state == 0) {
            for (int r = 1; r < NCTA; ++r) {
                Smem *R = cluster.map_shared_rank(&S, r);
                for (int b = tid; b < 6 * n; b += THREADS) {
                    const int c = b / n, k = b - c * n;
                    R->Y[c][k] = S.Y[c][k];
                }
            }
        }
        __threadfence();
        __syncthreads();
        if (tid == 0) {
            for (int r = 0; r < NCTA; ++r) {
                Smem *R = cluster.map_shared_rank(&S, r);
                R->rec_H = H; R->rec_state = next_state;
            }
            __threadfence();
            for (int r = 0; r < NCTA; ++r) cluster.map_shared_rank(&S, r)->seq_end = ns;
        }
        BC_PROF(4)
    }
#ifdef GENGA_BC_PROF
    if (master && tid == 0 && nsteps) { for (int k = 0; k < 5; ++k) nsteps[2 + k] = (int)(pf_acc[k] >> 4); }
#endif
    return ok;
}

}  // namespace genga
