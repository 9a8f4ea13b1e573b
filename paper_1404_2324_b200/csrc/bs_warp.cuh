// Bulirsch-Stoer for one SMALL close-encounter group (2..8 bodies) on ONE WARP (PAPER.md L116,
// L286-314; the paper's Table 3, gives groups of 2 a block of 4 threads).
//
// Most groups are pairs and triples (cfg1: 140 of 165 groups; cfg2, cfg3, cfg4: nearly all), and what a
// group costs is the LENGTH of its dependent chain: an attempted step of the sequential algorithm
// is 1 + 2 + 4 + ... + 2(k+1) force evaluations one after the other.  Here the eight
// modified-midpoint runs (n_k = 2, 4, ..., 16 substeps, all from the same state) sit side by side
// in the lanes of one warp:
//     S = 2 (pairs), S = 4 (groups of 3, 4):  lane = S c + b  integrates column c (8 columns) of
//                              body b, 16 force evaluations per attempt;
//     S = 8 (groups of 5..8):  lane = 8 g + b  integrates columns g and 7 - g (18 substeps each) of
//                              body b, 18 force evaluations per attempt.
// A lane keeps its body's midpoint state in registers; the positions of the other bodies of the
// SAME column come by segmented shuffles (no shared memory, no barrier on the chain).  Column
// results go to a small per-warp shared tableau; the lanes of the first segment run the
// Aitken-Neville recurrence row by row and take the first row k* whose error passes -- exactly the
// row the sequential algorithm stops at, so the accepted state is the same; columns beyond k* are
// speculative work of lanes that would otherwise idle.
#pragma once
#include "bs.cuh"

namespace genga {

constexpr int BW_MAXN = 8;          // largest group of the warp layout
constexpr int BW_WARPS = 4;         // warps per block: one per SM sub-partition

struct BwSmem {
    double tab[BS_KMAX][6][BW_MAXN];     // column results T[k][0], then the diagonal T[k][k]
};

// Forces on this lane's body at TWO positions qA, qB at once; the partners are the other lanes of its
// S-lane segment (same column): partner t = 0..n-2 sits in segment lane src[t] = (b + 1 + t) mod n and
// carries rcij[t] = max(rc_b, rc_j) (0 for a massless or missing partner, so that it never passes the
// test), irc[t] = 1 / (0.9 rcij), gm[t] = G m_j.  Star fixed at the origin (L314); every pair of the group
// is examined at every evaluation (L505).
// Why two: in Gragg's rule q_{k+1} = q_{k-1} + 2 eta V_k and V_{k+1} = V_{k-1} + 2 eta a(q_k), so a(q_k)
// and a(q_{k+1}) do not depend on each other; evaluated in one straight-line block their two dependent
// chains (~300 cycles each: shuffle, distance, changeover weight) overlap.  For S <= 4 there is no branch
// at all (a partner outside rc_ij is computed and discarded); for S = 8 a partner nobody in the warp is
// close to is skipped.
template <int S>
__device__ __forceinline__ void bw_rhs2(const double (&qA)[3], const double (&qB)[3], double Gm0, const int (&src)[S],
                                        const double (&rcij)[S], const double (&irc)[S], const double (&gm)[S],
                                        double (&aA)[3], double (&aB)[3])
{
    GENGA_BS_RHS_HOOK();
    const unsigned full = 0xffffffffu;
    double rA = fma(qA[2], qA[2], fma(qA[1], qA[1], qA[0] * qA[0]));
    double rB = fma(qB[2], qB[2], fma(qB[1], qB[1], qB[0] * qB[0]));
    double sA = -Gm0 * rinv3_fast(rA), sB = -Gm0 * rinv3_fast(rB);
    double ax = sA * qA[0], ay = sA * qA[1], az = sA * qA[2];
    double bx = sB * qB[0], by = sB * qB[1], bz = sB * qB[2];
#pragma unroll
    for (int t = 0; t < S - 1; ++t) {
        double dxA = __shfl_sync(full, qA[0], src[t], S) - qA[0];
        double dyA = __shfl_sync(full, qA[1], src[t], S) - qA[1];
        double dzA = __shfl_sync(full, qA[2], src[t], S) - qA[2];
        double dxB = __shfl_sync(full, qB[0], src[t], S) - qB[0];
        double dyB = __shfl_sync(full, qB[1], src[t], S) - qB[1];
        double dzB = __shfl_sync(full, qB[2], src[t], S) - qB[2];
        double dA = fma(dzA, dzA, fma(dyA, dyA, dxA * dxA)), dB = fma(dzB, dzB, fma(dyB, dyB, dxB * dxB));
        const double rc2 = rcij[t] * rcij[t];
        bool inA = dA < rc2, inB = dB < rc2;
        if (S <= 4 || __any_sync(full, inA || inB)) {             // S = 8: warp-uniform skip
            double scA = direct_scale_nb(inA ? dA : 1.0, rcij[t], irc[t], gm[t]);
            double scB = direct_scale_nb(inB ? dB : 1.0, rcij[t], irc[t], gm[t]);
            scA = inA ? scA : 0.0; scB = inB ? scB : 0.0;
            ax = fma(scA, dxA, ax); ay = fma(scA, dyA, ay); az = fma(scA, dzA, az);
            bx = fma(scB, dxB, bx); by = fma(scB, dyB, by); bz = fma(scB, dzB, bz);
        }
    }
    aA[0] = ax; aA[1] = ay; aA[2] = az;
    aB[0] = bx; aB[1] = by; aB[2] = bz;
}

// The same for the 8-lane segments (groups of 5..8 bodies), in two phases so that the expensive changeover
// weight is evaluated once per close pair instead of once per partner slot: (1) squared distances to the
// n - 1 partners at both points, one bit per partner that is inside rc_ij at either point; (2) while any
// lane has a bit left, every lane takes ITS next close partner (a shuffle with a per-lane source), evaluates
// both weights and accumulates.  Rounds = the largest number of close partners of any body (typically 1 or 2).
__device__ __forceinline__ void bw_rhs2_seg8(const double (&qA)[3], const double (&qB)[3], const int n, const int b,
                                             double Gm0, double G, double my_rc, double my_m, const double (&rcij)[8],
                                             double (&aA)[3], double (&aB)[3])
{
    GENGA_BS_RHS_HOOK();
    const unsigned full = 0xffffffffu;
    double rA = fma(qA[2], qA[2], fma(qA[1], qA[1], qA[0] * qA[0]));
    double rB = fma(qB[2], qB[2], fma(qB[1], qB[1], qB[0] * qB[0]));
    double sA = -Gm0 * rinv3_fast(rA), sB = -Gm0 * rinv3_fast(rB);
    double ax = sA * qA[0], ay = sA * qA[1], az = sA * qA[2];
    double bx = sB * qB[0], by = sB * qB[1], bz = sB * qB[2];
    unsigned close = 0u;
#pragma unroll
    for (int t = 0; t < 7; ++t) {
        if (t < n - 1) {                                          // warp-uniform
            int j = b + 1 + t;
            j = j >= n ? j - n : j;
            double dxA = __shfl_sync(full, qA[0], j, 8) - qA[0], dyA = __shfl_sync(full, qA[1], j, 8) - qA[1], dzA = __shfl_sync(full, qA[2], j, 8) - qA[2];
            double dxB = __shfl_sync(full, qB[0], j, 8) - qB[0], dyB = __shfl_sync(full, qB[1], j, 8) - qB[1], dzB = __shfl_sync(full, qB[2], j, 8) - qB[2];
            double dA = fma(dzA, dzA, fma(dyA, dyA, dxA * dxA)), dB = fma(dzB, dzB, fma(dyB, dyB, dxB * dxB));
            const double rc2 = rcij[t] * rcij[t];
            if (fmin(dA, dB) < rc2) close |= 1u << t;
        }
    }
    while (__any_sync(full, close != 0u)) {
        const bool act = close != 0u;
        const int t = act ? __ffs(close) - 1 : 0;
        close &= close - 1;
        int j = b + 1 + t;
        j = j >= n ? j - n : j;
        j = act ? j : b;
        double dxA = __shfl_sync(full, qA[0], j, 8) - qA[0], dyA = __shfl_sync(full, qA[1], j, 8) - qA[1], dzA = __shfl_sync(full, qA[2], j, 8) - qA[2];
        double dxB = __shfl_sync(full, qB[0], j, 8) - qB[0], dyB = __shfl_sync(full, qB[1], j, 8) - qB[1], dzB = __shfl_sync(full, qB[2], j, 8) - qB[2];
        const double rcj = __shfl_sync(full, my_rc, j, 8), mj = __shfl_sync(full, my_m, j, 8);
        const double r = fmax(my_rc, rcj), rc2 = r * r;
        double dA = fma(dzA, dzA, fma(dyA, dyA, dxA * dxA)), dB = fma(dzB, dzB, fma(dyB, dyB, dxB * dxB));
        const bool inA = act && dA < rc2, inB = act && dB < rc2;
        const double ir = rcp_fast(0.9 * (act ? r : 1.0)), gmj = G * mj;
        double scA = direct_scale_nb(inA ? dA : 1.0, r, ir, gmj), scB = direct_scale_nb(inB ? dB : 1.0, r, ir, gmj);
        scA = inA ? scA : 0.0; scB = inB ? scB : 0.0;
        ax = fma(scA, dxA, ax); ay = fma(scA, dyA, ay); az = fma(scA, dzA, az);
        bx = fma(scB, dxB, bx); by = fma(scB, dyB, by); bz = fma(scB, dzB, bz);
    }
    aA[0] = ax; aA[1] = ay; aA[2] = az;
    aB[0] = bx; aB[1] = by; aB[2] = bz;
}

// One entry of the Aitken-Neville tableau in (H/n_k)^2: component c of body b.  Reads the column results
// T[k][0], writes the diagonal T[k][k] back and returns the squared last corrections (T[k][k] - T[k][k-1])^2.
__device__ __forceinline__ void bw_neville(BwSmem &W, int c, int b, double (&d2)[BS_KMAX])
{
    // column by column, rows from the bottom up, in place: T[k] <- T[k][j] = T[k][j-1] + (T[k][j-1] - T[k-1][j-1]) / ((n_k / n_{k-j})^2 - 1).
    // The updates of one column are independent of each other, so the dependent chain is 7 steps, not 28.
    double T[BS_KMAX];
#pragma unroll
    for (int k = 0; k < BS_KMAX; ++k) { T[k] = W.tab[k][c][b]; d2[k] = 0.0; }
#pragma unroll
    for (int j = 1; j < BS_KMAX; ++j) {
#pragma unroll
        for (int k = BS_KMAX - 1; k >= j; --k) {
            const double ratio = double(k + 1) / double(k - j + 1);
            const double iden = 1.0 / (ratio * ratio - 1.0);
            const double nxt = T[k] + (T[k] - T[k - 1]) * iden;
            if (k == j) { const double diff = nxt - T[k]; d2[k] = diff * diff; }
            T[k] = nxt;
        }
    }
#pragma unroll
    for (int k = 0; k < BS_KMAX; ++k) W.tab[k][c][b] = T[k];      // T[k][k]
}

// Integrate one group over h.  Lane = S * g + b; Y = state of body b (same in every segment; any
// finite dummy for b >= n).  On return Y holds the result.  Returns false on step-size underflow
// (uniform over the warp).
template <int S>
__device__ __forceinline__ bool bw_integrate(BwSmem &W, const int lane, const int n, const double Gm0, const double my_rc,
                                             const double my_m, const double G, double (&Y)[6], const double h,
                                             const double eps, int *nsteps)
{
    constexpr int NCG = 32 / S;                // segments: 16 (8 of them idle), 8 or 4
    constexpr int CPL = NCG >= BS_KMAX ? 1 : BS_KMAX / NCG;          // columns per lane: 1 or 2
    constexpr int NIT = CPL == 1 ? BS_KMAX : BS_KMAX + 1;            // double force evaluations per attempt
    constexpr int NROUND = (6 * S + 31) / 32;                         // tableau entries (c, b) per lane
    const unsigned full = 0xffffffffu;
    const int cg = lane / S, b = lane % S;
    const bool body = b < n && cg < BS_KMAX;

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
    double q[3], V[3], acc0[3], isq = 0.0, isv = 0.0;
    while (!last) {
        double rem = h - done;
        if (fabs(H) >= fabs(rem)) { H = rem; last = true; }
        if (fresh) {
#pragma unroll
            for (int c = 0; c < 3; ++c) { q[c] = Y[c]; V[c] = Y[3 + c]; }
            isq = body ? 1.0 / (q[0] * q[0] + q[1] * q[1] + q[2] * q[2]) : 0.0;
            isv = body ? 1.0 / (V[0] * V[0] + V[1] * V[1] + V[2] * V[2]) : 0.0;
            double dummy[3];
            if constexpr (S == 8) bw_rhs2_seg8(q, q, n, b, Gm0, G, my_rc, my_m, rcij, acc0, dummy);
            else bw_rhs2<S>(q, q, Gm0, src, rcij, irc, gm, acc0, dummy);
            fresh = false;
        }
        // ---- my column(s): Gragg's modified midpoint rule, two substeps per iteration, all lanes in step.
        // Column col (n_k = 2 (col + 1) substeps) ends in its iteration number col.
        int col = cg, left = col + 1, pass = 0;
        double eta = H / (2 * (col + 1));
        double qa[3], Va[3], qb[3], Vb[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            qa[c] = q[c]; Va[c] = V[c];
            qb[c] = q[c] + eta * V[c]; Vb[c] = V[c] + eta * acc0[c];
        }
#pragma unroll 1
        for (int it = 0; it < NIT; ++it) {
            double qc[3], A[3], C[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) qc[c] = qa[c] + 2.0 * eta * Vb[c];
            if constexpr (S == 8) bw_rhs2_seg8(qb, qc, n, b, Gm0, G, my_rc, my_m, rcij, A, C);
            else bw_rhs2<S>(qb, qc, Gm0, src, rcij, irc, gm, A, C);
            const bool fin = --left == 0;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                double vc = Va[c] + 2.0 * eta * A[c];
                if (fin && body) {
                    W.tab[col][c][b] = 0.5 * (qc[c] + qb[c] + eta * vc);
                    W.tab[col][3 + c][b] = 0.5 * (vc + Vb[c] + eta * C[c]);
                }
                double qd = qb[c] + 2.0 * eta * vc, vd = Vb[c] + 2.0 * eta * C[c];
                qa[c] = qc[c]; Va[c] = vc; qb[c] = qd; Vb[c] = vd;
            }
            if (CPL == 2 && fin && pass == 0) {                       // second column of this lane
                pass = 1; col = BS_KMAX - 1 - cg; left = col + 1; eta = H / (2 * (col + 1));
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    qa[c] = q[c]; Va[c] = V[c];
                    qb[c] = q[c] + eta * V[c]; Vb[c] = V[c] + eta * acc0[c];
                }
            } else if (left < 0) {                                    // finished lanes: stay at a harmless point
#pragma unroll
                for (int c = 0; c < 3; ++c) { qa[c] = q[c]; qb[c] = q[c]; Va[c] = 0.0; Vb[c] = 0.0; }
                eta = 0.0;
            }
        }
        __syncwarp();
        // ---- Aitken-Neville tableau in (H/n_k)^2, one (component, body) entry per lane; first row whose error passes
        double d2[NROUND][BS_KMAX];
#pragma unroll
        for (int r = 0; r < NROUND; ++r) {
            const int item = lane + 32 * r, c = item / S, bb = item % S;
#pragma unroll
            for (int k = 0; k < BS_KMAX; ++k) d2[r][k] = 0.0;
            if (item < 6 * S && bb < n) bw_neville(W, c, bb, d2[r]);
        }
        int kstar = -1;
#pragma unroll
        for (int k = BS_KMAX - 1; k >= 1; --k) {
            // body b (lanes < S): sum over the components, entry (c, b) sits in lane (c S + b) % 32 of round (c S + b) / 32
            double dq = 0.0, dv = 0.0;
#pragma unroll
            for (int c = 0; c < 6; ++c) {
                const int item = c * S + (lane % S);
                double v = __shfl_sync(full, d2[(c * S) / 32][k], item & 31);
                if (c < 3) dq += v; else dv += v;
            }
            double r = (lane < S && body) ? fmax(dq * isq, dv * isv) : 0.0;
#pragma unroll
            for (int o = S / 2; o > 0; o >>= 1) r = fmax(r, __shfl_xor_sync(full, r, o, S));
            if (r <= eps2) kstar = k;
        }
        kstar = __shfl_sync(full, kstar, 0);
        __syncwarp();
        if (kstar >= 0) {
            if (body) {
#pragma unroll
                for (int c = 0; c < 6; ++c) Y[c] = W.tab[kstar][c][b];
            }
            __syncwarp();
            done += H;
            if (nsteps) ++nsteps[0];
            if (kstar <= 4) H *= 1.5;
            fresh = true;
        } else {
            H *= 0.5; last = false;
            if (nsteps) ++nsteps[1];
            if (fabs(H) < BS_HMIN * fabs(h)) return false;
        }
    }
    return true;
}

}  // namespace genga
