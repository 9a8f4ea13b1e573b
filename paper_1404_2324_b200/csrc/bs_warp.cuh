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

// G m_j (1 - W(d, rc_ij)) / d^3 as direct_scale(), without a branch (all lanes of a warp run it
// together; `in` selects afterwards).
__device__ __forceinline__ double direct_scale_nb(double d2, double rcij, double irc09, double Gmj)
{
    double rinv = rsqrt_fast(d2);
    double dd = d2 * rinv;
    double y = (dd - 0.1 * rcij) * irc09;
    double D = fma(2.0 * y, y - 1.0, 1.0);                    // >= 1/2 for every y
    double iD = rcp_fast(D);
    double yD = y * iD;                                       // K = y yD
    double dK = 2.0 * (1.0 - y) * (yD * iD) * irc09;
    double w1 = 1.0 - fma(y, yD, -dd * dK);
    w1 = y > 0.0 ? w1 : 1.0;
    return Gmj * (rinv * rinv) * rinv * w1;
}

// Force on this lane's body at position q; the partners are the other lanes of its S-lane segment
// (same column): partner t = 0..n-2 sits in segment lane src[t] = (b + 1 + t) mod n and carries
// rcij[t] = max(rc_b, rc_j) (0 for a massless or missing partner, so that it never passes the test),
// irc[t] = 1 / (0.9 rcij), gm[t] = G m_j.  n is uniform over the warp.
// Star fixed at the origin (L314); every pair of the group is examined at every evaluation (L505).
template <int S>
__device__ __forceinline__ void bw_rhs(const double q[3], const int n, double Gm0, const int (&src)[S], const double (&rcij)[S],
                                       const double (&irc)[S], const double (&gm)[S], double a[3])
{
    GENGA_BS_RHS_HOOK();
    const unsigned full = 0xffffffffu;
    double r2 = fma(q[2], q[2], fma(q[1], q[1], q[0] * q[0]));
    double s0 = -Gm0 * rinv3_fast(r2);
    double ax = s0 * q[0], ay = s0 * q[1], az = s0 * q[2];
#pragma unroll
    for (int t = 0; t < S - 1; ++t) {
        if (t < n - 1) {                                      // warp-uniform
            double dx = __shfl_sync(full, q[0], src[t], S) - q[0];
            double dy = __shfl_sync(full, q[1], src[t], S) - q[1];
            double dz = __shfl_sync(full, q[2], src[t], S) - q[2];
            double d2 = fma(dz, dz, fma(dy, dy, dx * dx));
            bool in = d2 < rcij[t] * rcij[t];
            if (__any_sync(full, in)) {                       // warp-uniform: no divergence
                double sc = direct_scale_nb(in ? d2 : 1.0, rcij[t], irc[t], gm[t]);
                sc = in ? sc : 0.0;
                ax = fma(sc, dx, ax); ay = fma(sc, dy, ay); az = fma(sc, dz, az);
            }
        }
    }
    a[0] = ax; a[1] = ay; a[2] = az;
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
    constexpr int NIT = CPL == 1 ? 2 * BS_KMAX : 2 * BS_KMAX + 2;   // force evaluations per attempt after the first
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
        bool valid = body && j != b && mj != 0.0 && r > 0.0;
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
            bw_rhs<S>(q, n, Gm0, src, rcij, irc, gm, acc0);
            fresh = false;
        }
        // ---- my column(s): Gragg's modified midpoint rule, all lanes in step
        int pass = 0, col = cg, nk = 2 * (col + 1), ms = 1;
        bool act = true;
        double eta = H / nk;
        double qa[3], Va[3], qb[3], Vb[3], acc[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            qa[c] = q[c]; Va[c] = V[c];
            qb[c] = q[c] + eta * V[c]; Vb[c] = V[c] + eta * acc0[c];
        }
#pragma unroll 1
        for (int it = 0; it < NIT; ++it) {
            bw_rhs<S>(qb, n, Gm0, src, rcij, irc, gm, acc);
            if (act) {
                if (ms < nk) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        double qn = qa[c] + 2.0 * eta * Vb[c];
                        double vn = Va[c] + 2.0 * eta * acc[c];
                        qa[c] = qb[c]; Va[c] = Vb[c]; qb[c] = qn; Vb[c] = vn;
                    }
                    ++ms;
                } else {
                    if (body) {
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            W.tab[col][c][b] = 0.5 * (qb[c] + qa[c] + eta * Vb[c]);
                            W.tab[col][3 + c][b] = 0.5 * (Vb[c] + Va[c] + eta * acc[c]);
                        }
                    }
                    if (++pass < CPL) {
                        col = BS_KMAX - 1 - cg; nk = 2 * (col + 1); ms = 1; eta = H / nk;
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            qa[c] = q[c]; Va[c] = V[c];
                            qb[c] = q[c] + eta * V[c]; Vb[c] = V[c] + eta * acc0[c];
                        }
                    } else {
                        act = false;
#pragma unroll
                        for (int c = 0; c < 3; ++c) qb[c] = q[c];      // idle lanes: keep evaluating a harmless point
                    }
                }
            }
        }
        __syncwarp();
        // ---- Aitken-Neville tableau in (H/n_k)^2 by the first segment; first row whose error passes
        double e[BS_KMAX];
#pragma unroll
        for (int k = 0; k < BS_KMAX; ++k) e[k] = 0.0;
        if (lane < S && body) {
            double dq2[BS_KMAX], dv2[BS_KMAX];
#pragma unroll
            for (int k = 0; k < BS_KMAX; ++k) { dq2[k] = 0.0; dv2[k] = 0.0; }
#pragma unroll
            for (int c = 0; c < 6; ++c) {
                double row[BS_KMAX] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
                for (int k = 0; k < BS_KMAX; ++k) {
                    double cur = W.tab[k][c][b], prev = row[0], diff = 0.0;
                    row[0] = cur;
#pragma unroll
                    for (int j = 1; j <= k; ++j) {
                        const double ratio = double(k + 1) / double(k - j + 1);
                        const double iden = 1.0 / (ratio * ratio - 1.0);
                        double tmp = row[j];
                        double nxt = cur + (cur - prev) * iden;
                        diff = nxt - cur;
                        cur = nxt;
                        row[j] = cur;
                        prev = tmp;
                    }
                    W.tab[k][c][b] = cur;                       // T[k][k]
                    if (c < 3) dq2[k] += diff * diff; else dv2[k] += diff * diff;
                }
            }
#pragma unroll
            for (int k = 1; k < BS_KMAX; ++k) e[k] = fmax(dq2[k] * isq, dv2[k] * isv);
        }
        int kstar = -1;
#pragma unroll
        for (int k = BS_KMAX - 1; k >= 1; --k) {
            double r = e[k];
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
            if (nsteps) ++*nsteps;
            if (kstar <= 4) H *= 1.5;
            fresh = true;
        } else {
            H *= 0.5; last = false;
            if (fabs(H) < BS_HMIN * fabs(h)) return false;
        }
    }
    return true;
}

}  // namespace genga
