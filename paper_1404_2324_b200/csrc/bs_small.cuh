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

struct BsmSmem {
    double tab[BSM_MAXL][BS_KMAX][6][BW_MAXN];   // [level][column][component][body]: column results T[k][0]
    double Y[6][BW_MAXN];                        // state at the start of the round / the accepted state
    double werr[BSM_MAXL][6][BW_MAXN];           // scaled squared corrections of the row under test
    int status[BSM_MAXL];                        // 0 running, 1 + k accepted at row k, -1 rejected, -2 step size underflow
};

// Integrate one group over h with NW warps (the whole block).  Lane layout as above; Y = state of body b = lane % S
// (any finite dummy for b >= n), the same in every segment.  On return Y holds the result in every lane.
// nsteps[0] += accepted steps, nsteps[1] += rejected attempts (as the sequential rule counts them).
template <int S, int NW>
__device__ __forceinline__ bool bsm_integrate(BsmSmem &W, const int n, const double Gm0, const double my_rc, const double my_m,
                                              const double G, double (&Y)[6], const double h, const double eps, int *nsteps)
{
    constexpr int SPW = 32 / S;                       // slots (columns) per warp
    constexpr int L = NW * SPW / BS_KMAX;             // speculation levels
    constexpr int LL = (8 * S < 32) ? 8 * S : 32;     // lanes of a level inside its first warp
    constexpr int NROUND = (6 * S + LL - 1) / LL;     // tableau entries (component, body) per checking lane
    static_assert(L >= 1 && L <= BSM_MAXL, "levels");
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

    double done = 0.0, H = h;
    bool last = false, fresh = true;
    const double eps2 = eps * eps;
    double q[3], V[3], acc0[3];
    double wsc[NROUND];                               // checker: 1 / |q_b|^2 or 1 / |V_b|^2 of its entries
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
            if constexpr (S == 8) bw_rhs2_seg8(q, q, n, b, Gm0, G, my_rc, my_m, rcij, acc0, dummy);
            else bw_rhs2<S>(q, q, Gm0, src, rcij, irc, gm, acc0, dummy);
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
        int winner = -1, wrow = 0;
        bool resolved = false;
#pragma unroll 1
        for (int it = 0; it < BS_KMAX && !resolved; ++it) {
            // ---- my column: Gragg's modified midpoint rule, two substeps per evaluation (bs_warp.cuh)
            const bool work = mystat == 0;            // my level is still undecided
            // warp-uniform: some column of this warp still runs
            if (__any_sync(full, work && it <= col)) {
                double qc[3], A[3], C[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) qc[c] = qa[c] + 2.0 * eta * Vb[c];
                if constexpr (S == 8) bw_rhs2_seg8(qb, qc, n, b, Gm0, G, my_rc, my_m, rcij, A, C);
                else bw_rhs2<S>(qb, qc, Gm0, src, rcij, irc, gm, A, C);
                const bool fin = it == col;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    double vc = Va[c] + 2.0 * eta * A[c];
                    if (fin && body && work) {
                        W.tab[lev][col][c][b] = 0.5 * (qc[c] + qb[c] + eta * vc);
                        W.tab[lev][col][3 + c][b] = 0.5 * (vc + Vb[c] + eta * C[c]);
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
            __syncthreads();
            // ---- the tableau row that became complete: T[it][j] = T[it][j-1] + (T[it][j-1] - T[it-1][j-1]) / ((n_it / n_{it-j})^2 - 1)
            if (checker && mystat == 0) {
                double wv[NROUND];
#pragma unroll
                for (int r = 0; r < NROUND; ++r) {
                    const int item = cl + LL * r, c = item / S, bb = item % S;
                    wv[r] = 0.0;
                    if (item < 6 * S && bb < n) {
                        double cur = W.tab[lev][it][c][bb], prev = prow[r][0], diff = 0.0;
                        prow[r][0] = cur;
#pragma unroll
                        for (int j = 1; j < BS_KMAX; ++j) {
                            if (j <= it) {
                                const double tmp = prow[r][j];
                                const double nxt = cur + (cur - prev) * c_bs_iden.v[it][j];
                                diff = nxt - cur;
                                cur = nxt;
                                prow[r][j] = cur;
                                prev = tmp;
                            }
                        }
                        wv[r] = diff * diff * wsc[r];
                        W.tab[lev][it][c][bb] = cur;              // T[it][it]: the state if this row is accepted
                        W.werr[lev][c][bb] = wv[r];
                    }
                }
            }
            __syncwarp();
            if (checker && mystat == 0 && it >= 1) {
                double e = 0.0;
                if (cl < n) {
                    const double dq = W.werr[lev][0][cl] + W.werr[lev][1][cl] + W.werr[lev][2][cl];
                    const double dv = W.werr[lev][3][cl] + W.werr[lev][4][cl] + W.werr[lev][5][cl];
                    e = fmax(dq, dv);
                }
                // the first S lanes of the level hold the bodies' errors
#pragma unroll
                for (int o = S / 2; o > 0; o >>= 1) e = fmax(e, __shfl_xor_sync(lmask, e, o, S));
                if (cl == 0) {
                    if (e <= eps2) W.status[lev] = 1 + it;
                    else if (it == BS_KMAX - 1) W.status[lev] = -1;
                }
            }
            if (it == 0 && checker && cl == 0) W.status[lev] = mystat;          // round start: running (or underflow)
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
        if (winner == -2) return false;
        if (winner >= 0) {
            if (body) {
#pragma unroll
                for (int c = 0; c < 6; ++c) Y[c] = W.tab[winner][wrow][c][b];
            }
            const double Hw = ldexp(H, -winner);
            done += Hw;
            H = Hw;
            if (nsteps) { ++nsteps[0]; nsteps[1] += winner; }
            if (wrow <= 4) H *= 1.5;
            if (winner > 0) last = false;
            fresh = true;
        } else {                                      // every level rejected
            if (nsteps) nsteps[1] += L;
            H = ldexp(H, -L); last = false;
            if (fabs(H) < BS_HMIN * fabs(h)) return false;
        }
        __syncthreads();                              // the tableau and the statuses may be overwritten
    }
    return true;
}

}  // namespace genga
