// Bulirsch-Stoer for one SMALL close-encounter group (2..8 bodies) on ONE THREAD BLOCK.
//
// What a group costs is the LENGTH of its dependent chain, and the step waits for the longest one.  Traces of the
// first layout (one warp per group, genga_bs_trace) showed where the chain goes: (i) a third of all attempted steps are
// REJECTED (all eight extrapolation columns fail, the step is halved: "first trial H = h; on failure H/2", DESIGN.md
// R-7), each a full chain of 8 double force evaluations thrown away; a deep encounter needs H = h/64 and pays six of
// them before its first accepted step; (ii) an accepted step mostly passes at row 2..4 of the tableau, but all eight
// columns were run to the end (8 evaluations instead of 3..5).  This layout removes both without changing a single
// accepted step:
//   * SPECULATION over the step size: the block integrates the attempts H, H/2, H/4, ... (L levels) side by side from
//     the same state.  The level taken is the first one, in that order, that passes -- exactly the step the sequential
//     rule arrives at after its rejections -- so the sequence of accepted steps (and with it the result) is the
//     sequential algorithm's; the rejected attempts cost no time any more.
//   * EARLY EXIT: column k (n_k = 2(k+1) substeps) finishes after k+1 evaluations; after every evaluation the tableau
//     row that has become complete is tested, and a level that passes at row k stops there (the row the sequential
//     algorithm stops at).
// A round (one accepted step) therefore costs k+1 evaluations if the largest step passes, 8 if it is rejected (its
// rejection is only known when its last column has failed).
//
// Lanes: S = 2, 4 or 8 lanes per column segment (bodies of one column, partners by segmented shuffles as in
// bs_warp.cuh); slot = warp * (32 / S) + lane / S, level = slot / 8, column = slot % 8.  A block of 4 warps takes a
// group of 2 bodies with S = 2 (8 levels), of 3..4 bodies with S = 4 (4 levels), of 5..8 bodies with S = 8 (2 levels,
// two warps per level: one column per lane).  The warps of a block meet at two block barriers per evaluation.
#pragma once
#include "bs_warp.cuh"

namespace genga {

constexpr int BSM_MAXL = 8;
constexpr int BSM_SLOTS = 16;        // levels x lanes per segment: 8 x 2, 4 x 4 or 2 x 8

struct BsmSmem {
    double tab[BS_KMAX][6][BSM_SLOTS];           // [column][component][level * S + body]: column results T[k][0], then T[k][k]
    double werr[BS_KMAX][6][BSM_SLOTS];          // scaled squared corrections of the rows under test
    double Y[6][BW_MAXN];                        // state at the start of the round
    int status[BSM_MAXL];                        // 0 running, 1 + k accepted at row k, -1 rejected, -2 step size underflow
    double R[BW_MAXN];                           // physical radii (collision test; < 0: none)
    int coll;                                    // look for collisions in every accepted step (L328)
    BwGroup8 grp;                                // S = 8: (rc, G m) of the bodies
    BwSlot8 slot[BSM_SLOTS];                     // S = 8: positions of each column segment (bw_rhs2_seg8)
};

// Does a pair of the group collide in the step just accepted (L328: the Hermite minimum of Eq. 10-12 over the step
// against (R_a + R_b)^2)?  Old state W.Y, new state row `wrow` of level `winner`.  The whole block; the same answer in
// every thread.  A group with a collision is handed to k_bs_generic, which integrates it again and merges the pair.
template <int S>
__device__ __noinline__ bool bsm_any_collision(BsmSmem &W, const int n, const int wrow, const int winner, const double H)
{
    int hit = 0;
    const int p = threadIdx.x;                   // pair number: (a, b), a < b < n <= 8: at most 28
    if (p < n * (n - 1) / 2) {
        int a = 0, rest = p;
        while (rest >= n - 1 - a) { rest -= n - 1 - a; ++a; }
        const int b = a + 1 + rest;
        if (W.R[a] >= 0.0 && W.R[b] >= 0.0) {
            double P0 = 0.0, Pd0 = 0.0, P1 = 0.0, Pd1 = 0.0;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double d0 = W.Y[c][b] - W.Y[c][a], w0 = W.Y[3 + c][b] - W.Y[3 + c][a];
                const double d1 = W.tab[wrow][c][winner * S + b] - W.tab[wrow][c][winner * S + a];
                const double w1 = W.tab[wrow][3 + c][winner * S + b] - W.tab[wrow][3 + c][winner * S + a];
                P0 += d0 * d0; Pd0 += 2.0 * d0 * w0; P1 += d1 * d1; Pd1 += 2.0 * d1 * w1;
            }
            hit = pair_collides(P0, P1, Pd0, Pd1, H, W.R[a] + W.R[b]) ? 1 : 0;
        }
    }
    return __syncthreads_or(hit) != 0;
}

// Integrate one group over h with NW warps (the whole block).  Lane layout as above; Y = state of body b = lane % S
// (any finite dummy for b >= n), the same in every segment.  On return Y holds the result in every lane.
// nsteps[0] += accepted steps, nsteps[1] += rejected attempts (as the sequential rule counts them).
//
// The tableau is not tested after every evaluation: a test costs about as much as two evaluations (two block barriers,
// a trip through shared memory, a reduction over the bodies).  It is tested when the row the previous step of this
// group was accepted at has become complete (row 4 at first), then every second row, and at the end; a test looks at all
// the rows completed since the last one and takes the FIRST that passes, so the accepted row is the sequential
// algorithm's whatever the schedule of the tests.
// Returns 0: step size underflow, 1: done, 2: a pair of the group collides (nothing written; see bsm_any_collision).
template <int S, int NW>
__device__ __forceinline__ int bsm_integrate(BsmSmem &W, const int n, const double Gm0, const double my_rc, const double my_m,
                                              const double G, double (&Y)[6], const double h, const double eps, int *nsteps)
{
    constexpr int SPW = 32 / S;                       // slots (columns) per warp
    constexpr int L = NW * SPW / BS_KMAX;             // speculation levels
    constexpr int LL = (8 * S < 32) ? 8 * S : 32;     // lanes of a level inside its first warp
    constexpr int NROUND = (6 * S + LL - 1) / LL;     // tableau entries (component, body) per checking lane
    static_assert(L >= 1 && L <= BSM_MAXL && L * S <= BSM_SLOTS, "levels");
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int slot = warp * SPW + lane / S, lev = slot / BS_KMAX, col = slot % BS_KMAX, b = lane % S;
    const bool body = b < n;
    // the lanes that test this level's tableau: the first LL lanes of the level (all in one warp)
    const int lfirst = (lev * BS_KMAX * S) & 31;      // first lane of my level in its first warp
    const bool checker = (S == 8 ? (warp & 1) == 0 : true) && lane >= lfirst && lane < lfirst + LL;
    const int cl = lane - lfirst;                     // 0 .. LL-1 for checkers
    const unsigned lmask = LL == 32 ? 0xffffffffu : (((1u << LL) - 1u) << lfirst);   // the checking lanes of my level

    int src[S];
    double rcij[S], irc[S], gm[S];
#pragma unroll
    for (int t = 0; t < S; ++t) {
        int j = b + 1 + t;
        j = j >= n ? j - n : j;
        j = body ? j : b;
        src[t] = j;
        double rcj = __shfl_sync(full, my_rc, j, S);
        double mj = __shfl_sync(full, my_m, j, S);
        double r = fmax(my_rc, rcj);
        bool valid = body && j != b && mj != 0.0 && r > 0.0 && t < n - 1;
        rcij[t] = valid ? r : 0.0;
        irc[t] = valid ? 1.0 / (0.9 * r) : 0.0;
        gm[t] = valid ? G * mj : 0.0;
    }

    // S = 8: FP32 pretest threshold of this body: positions stay within Q = 2 max_b(|q_b| + |h| |V_b|) (max norms) of the
    // origin during the step, so rounding them to FP32 moves a separation by < 2^-22 Q and the FP32 evaluation of its
    // square adds < 2^-21 relative: thr = (rc + 2^-20 Q)^2 (1 + 2^-18) (as bs_cluster.cuh); bodies without mass exert no
    // force and are left out of everybody's partner mask.
    float thr = 0.f;
    unsigned massive = 0u;
    BwSlot8 &myslot = W.slot[slot % BSM_SLOTS];
    if constexpr (S == 8) {
        double qm = body ? fmax(fmax(fabs(Y[0]), fabs(Y[1])), fabs(Y[2])) + fabs(h) * fmax(fmax(fabs(Y[3]), fabs(Y[4])), fabs(Y[5])) : 0.0;
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) qm = fmax(qm, __shfl_xor_sync(full, qm, o, 8));
        const double w = my_rc + 0x1.0p-20 * 2.0 * qm;
        thr = body ? __double2float_ru(w * w * (1.0 + 0x1.0p-18)) : 0.f;
        massive = __ballot_sync(full, body && my_m != 0.0);
        massive = (massive >> (lane & 24)) & 0xffu;               // the eight lanes of my segment
        if (warp == 0 && lane < 8) W.grp.rcm[lane] = make_double2(body ? my_rc : 0.0, body ? G * my_m : 0.0);
        __syncthreads();
    }

    double done = 0.0, H = h;
    bool last = false, fresh = true;
    const double eps2 = eps * eps;
    double q[3], V[3], acc0[3];
    double wsc[NROUND];                               // checker: 1 / |q_b|^2 or 1 / |V_b|^2 of its entries
    int hint = 4;                                     // the row to test first
    while (!last) {
        double rem = h - done;
        if (fabs(rem) <= 8.0 * 2.220446049250313e-16 * fabs(h)) break;     // a remainder of a few ulp of h: done
        if (fabs(H) >= fabs(rem)) { H = rem; last = true; }
        if (fresh) {
#pragma unroll
            for (int c = 0; c < 3; ++c) { q[c] = Y[c]; V[c] = Y[3 + c]; }
            if (warp == 0 && lane < S && body) {
#pragma unroll
                for (int c = 0; c < 6; ++c) W.Y[c][b] = Y[c];
            }
            double dummy[3];
            if constexpr (S == 8) bw_rhs2_seg8(W.grp, myslot, q, q, n, b, Gm0, my_rc, thr, massive, acc0, dummy);
            else bw_rhs2<S>(q, q, Gm0, src, rcij, irc, gm, n, acc0, dummy);
            __syncthreads();
            if (checker) {
#pragma unroll
                for (int r = 0; r < NROUND; ++r) {
                    const int item = cl + LL * r, c = item / S, bb = item % S;
                    wsc[r] = 0.0;
                    if (item < 6 * S && bb < n) {
                        const int o = c < 3 ? 0 : 3;
                        const double s2 = W.Y[o][bb] * W.Y[o][bb] + W.Y[o + 1][bb] * W.Y[o + 1][bb] + W.Y[o + 2][bb] * W.Y[o + 2][bb];
                        wsc[r] = 1.0 / s2;
                    }
                }
            }
            fresh = false;
        }
        // ---- one round: level l attempts H / 2^l
        const double Hl = ldexp(H, -lev);
        const bool under = lev > 0 && fabs(Hl) < BS_HMIN * fabs(h);
        double eta = Hl / (2 * (col + 1));
        double qa[3], Va[3], qb[3], Vb[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            qa[c] = q[c]; Va[c] = V[c];
            qb[c] = q[c] + eta * V[c]; Vb[c] = V[c] + eta * acc0[c];
        }
        int mystat = under ? -2 : 0;                  // status of my level as this lane knows it
        double prow[NROUND][BS_KMAX];                 // checker: the previous tableau row T[k-1][0..k-1] of its entries
#pragma unroll
        for (int r = 0; r < NROUND; ++r)
#pragma unroll
            for (int j = 0; j < BS_KMAX; ++j) prow[r][j] = 0.0;
        if (checker && cl == 0) W.status[lev] = mystat;           // read after the barriers of the first test
        int winner = -1, wrow = 0, tested = -1, next_test = hint;
        bool resolved = false;
#pragma unroll 1
        for (int it = 0; it < BS_KMAX && !resolved; ++it) {
            // ---- my column: Gragg's modified midpoint rule, two substeps per evaluation (bs_warp.cuh)
            const bool work = mystat == 0;            // my level is still undecided
            if (__any_sync(full, work && it <= col)) {            // warp-uniform: some column of this warp still runs
                double qc[3], A[3], C[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) qc[c] = qa[c] + 2.0 * eta * Vb[c];
                if constexpr (S == 8) bw_rhs2_seg8(W.grp, myslot, qb, qc, n, b, Gm0, my_rc, thr, massive, A, C);
                else bw_rhs2<S>(qb, qc, Gm0, src, rcij, irc, gm, n, A, C);
                const bool fin = it == col;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    double vc = Va[c] + 2.0 * eta * A[c];
                    if (fin && body && work) {
                        W.tab[col][c][lev * S + b] = 0.5 * (qc[c] + qb[c] + eta * vc);
                        W.tab[col][3 + c][lev * S + b] = 0.5 * (vc + Vb[c] + eta * C[c]);
                    }
                    double qd = qb[c] + 2.0 * eta * vc, vd = Vb[c] + 2.0 * eta * C[c];
                    qa[c] = qc[c]; Va[c] = vc; qb[c] = qd; Vb[c] = vd;
                }
                if (it >= col) {                      // finished lanes: stay at a harmless point
#pragma unroll
                    for (int c = 0; c < 3; ++c) { qa[c] = q[c]; qb[c] = q[c]; Va[c] = 0.0; Vb[c] = 0.0; }
                    eta = 0.0;
                }
            }
            if (it < next_test && it < BS_KMAX - 1) continue;     // no test after this evaluation (uniform over the block)
            __syncthreads();
            // ---- the tableau rows completed since the last test: T[r][j] = T[r][j-1] + (T[r][j-1] - T[r-1][j-1]) / ((n_r / n_{r-j})^2 - 1)
            if (checker && mystat == 0) {
#pragma unroll 1
                for (int row = tested + 1; row <= it; ++row) {
#pragma unroll
                    for (int r = 0; r < NROUND; ++r) {
                        const int item = cl + LL * r, c = item / S, bb = item % S;
                        if (item < 6 * S && bb < n) {
                            double cur = W.tab[row][c][lev * S + bb], prev = prow[r][0], diff = 0.0;
                            prow[r][0] = cur;
#pragma unroll
                            for (int j = 1; j < BS_KMAX; ++j) {
                                if (j <= row) {
                                    const double tmp = prow[r][j];
                                    const double nxt = cur + (cur - prev) * c_bs_iden.v[row][j];
                                    diff = nxt - cur;
                                    cur = nxt;
                                    prow[r][j] = cur;
                                    prev = tmp;
                                }
                            }
                            W.tab[row][c][lev * S + bb] = cur;    // T[row][row]: the state if this row is accepted
                            W.werr[row][c][lev * S + bb] = diff * diff * wsc[r];
                        }
                    }
                }
            }
            __syncwarp();
            if (checker && mystat == 0) {
                int pass = -1;                        // first row, among the new ones, whose error passes
#pragma unroll 1
                for (int row = max(tested + 1, 1); row <= it; ++row) {
                    double e = 0.0;
                    if (cl < n) {
                        const double dq = W.werr[row][0][lev * S + cl] + W.werr[row][1][lev * S + cl] + W.werr[row][2][lev * S + cl];
                        const double dv = W.werr[row][3][lev * S + cl] + W.werr[row][4][lev * S + cl] + W.werr[row][5][lev * S + cl];
                        e = fmax(dq, dv);
                    }
#pragma unroll
                    for (int o = S / 2; o > 0; o >>= 1) e = fmax(e, __shfl_xor_sync(lmask, e, o, S));   // the first S lanes of the level hold the bodies' errors
                    e = __shfl_sync(lmask, e, lfirst);
                    if (pass < 0 && e <= eps2) pass = row;
                }
                if (cl == 0) {
                    if (pass >= 0) W.status[lev] = 1 + pass;
                    else if (it == BS_KMAX - 1) W.status[lev] = -1;
                }
            }
            tested = it;
            next_test = min(it + 2, BS_KMAX - 1);
            __syncthreads();
            // ---- decision, the same in every thread: the first level, in the order H, H/2, ..., that passed
            mystat = W.status[lev];
#pragma unroll
            for (int l = 0; l < L; ++l) {
                if (resolved) break;
                const int st = W.status[l];
                if (st > 0) { winner = l; wrow = st - 1; resolved = true; }
                else if (st == 0) break;              // still running: the levels behind it have to wait
                else if (st == -2) { resolved = true; winner = -2; }
            }
        }
        if (winner == -2) return 0;
        if (winner >= 0) {
            if (W.coll && bsm_any_collision<S>(W, n, wrow, winner, ldexp(H, -winner))) return 2;
            if (body) {
#pragma unroll
                for (int c = 0; c < 6; ++c) Y[c] = W.tab[wrow][c][winner * S + b];
            }
            const double Hw = ldexp(H, -winner);
            done += Hw;
            H = Hw;
            if (nsteps) { ++nsteps[0]; nsteps[1] += winner; }
            if (wrow <= 4) H *= 1.5;
            if (winner > 0) last = false;
            fresh = true;
            hint = max(2, wrow);
        } else {                                      // every level rejected
            if (nsteps) nsteps[1] += L;
            H = ldexp(H, -L); last = false;
            if (fabs(H) < BS_HMIN * fabs(h)) return 0;
        }
        __syncthreads();                              // the tableau and the statuses may be overwritten
    }
    return 1;
}

}  // namespace genga
