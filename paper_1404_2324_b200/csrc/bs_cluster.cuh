// Bulirsch-Stoer for one close-encounter group on a thread-block CLUSTER.
//
// The cost of Bulirsch-Stoer on a GPU is latency, not arithmetic: one step is a chain of
// 2 + 4 + ... + 2(k+1) dependent force evaluations, each a dependent FP64 chain of ~25 operations,
// and cfg1 has only ~165 groups per time step.  The paper parallelises inside one force
// evaluation (p threads per body, Table 3).  Here the extrapolation COLUMNS run side by
// side as well: the modified-midpoint runs with n_k = 2, 4, ..., 16 substeps all start from the same
// state, so the CTAs of a cluster of CS integrate 8 / CS columns each (paired so that every CTA
// does the same number of substeps: CS = 4 takes columns {r, 7 - r}, 18 substeps each) in their own
// shared memory, and the chain per attempted step shrinks from 72 force evaluations to 17 (CS = 8)
// or 19 (CS = 4).  Column results go to CTA 0 through distributed shared memory; CTA 0 fills the
// Aitken-Neville tableau row by row, takes the first row k* whose error passes (exactly the
// row the sequential algorithm stops at, so the result is the same), and every CTA
// picks the new state up from CTA 0.  Columns beyond k* are speculative work on otherwise idle SMs.
//
// Inside a CTA, body i owns L adjacent lanes (a power of two, at most a warp); lane s of the
// segment takes partners j = s, s+L, ... and the star as partner j = n; the segment sum is an
// xor-butterfly (fixed order); lane 0 of the segment ("owner") carries the body's midpoint
// state in registers.  Positions are exchanged through a double-buffered shared array: one
// __syncthreads per force evaluation.
#pragma once
#include <cooperative_groups.h>

#include "bs.cuh"

namespace genga {

namespace cg = cooperative_groups;

template <int MAXN, int THREADS>
struct BcSmem {
    double pos[2][2][3][MAXN];      // [buffer][point A / B][component][body]
    float4 pf[2][2][MAXN];          // positions rounded to FP32 for the conservative pretest, .w = thr2: one LDS.128 per partner
    double isq[MAXN], isv[MAXN];    // 1 / |q|^2, 1 / |V|^2 at the start of the attempted step (error norm)
    float thr2[MAXN];               // (rc_i + margin)^2 rounded up
    double m[MAXN], rc[MAXN], irc[MAXN];
    double Y[6][MAXN];              // state at the start of the attempted step
    double tab[BS_KMAX][6][MAXN];   // CTA 0: column results T[k][0], then the diagonal T[k][k]
    double wmax[THREADS / 32][BS_KMAX];
    double red[THREADS / 32];
    int cur, kstar;
};

struct BcLane {
    int n, L, i, s;
    bool owner;
};

template <int THREADS>
__device__ __forceinline__ BcLane bc_lanes(int n)
{
    int P = 2, Q = 2;
    while (P < n) P <<= 1;              // bodies, rounded up to a power of two
    while (Q < n + 1) Q <<= 1;          // partners of a body (the others + the star)
    BcLane t;
    t.n = n; t.L = min(min(32, THREADS / P), Q);
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
template <int MAXN, int THREADS>
__device__ __forceinline__ void bc_rhs2(BcSmem<MAXN, THREADS> &S, const BcLane &t, int &buf, double G, double m0,
                                        const double qA[3], const double qB[3], double aA[3], double aB[3])
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
    __syncthreads();
    buf ^= 1;
    double ax = 0.0, ay = 0.0, az = 0.0, bx = 0.0, by = 0.0, bz = 0.0;
    if (t.i < t.n) {
        const int n = t.n, L = t.L, i = t.i;
        const float4 mA = fA[i], mB = fB[i];
        const float ft = mA.w;
        const double xA = pA[0][i], yA = pA[1][i], zA = pA[2][i], xB = pB[0][i], yB = pB[1][i], zB = pB[2][i];
        const double my_rc = S.rc[i], my_irc = S.irc[i];
        for (int j0 = t.s; j0 <= n; j0 += 32 * L) {              // partner j = n is the star
            unsigned mask = 0u;
#pragma unroll 4
            for (int kk = 0; kk < 32; ++kk) {
                int j = j0 + kk * L;
                if (j > n) break;
                int jc = j < n ? j : i;                           // star / self: computed, not used
                const float4 pa = fA[jc], pb = fB[jc];
                float dx = pa.x - mA.x, dy = pa.y - mA.y, dz = pa.z - mA.z;
                float ex = pb.x - mB.x, ey = pb.y - mB.y, ez = pb.z - mB.z;
                float d2 = fminf(fmaf(dz, dz, fmaf(dy, dy, dx * dx)), fmaf(ez, ez, fmaf(ey, ey, ex * ex)));
                bool in = d2 < fmaxf(ft, pa.w) && j != i && j != n;
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
        // the star (fixed at the origin): every lane of the body computes it, lane 0 keeps it (no split of the warp)
        {
            double rA = xA * xA + yA * yA + zA * zA, rB = xB * xB + yB * yB + zB * zB;
            double sA = -G * m0 * rinv3_fast(rA), sB = -G * m0 * rinv3_fast(rB);
            sA = t.s == 0 ? sA : 0.0; sB = t.s == 0 ? sB : 0.0;
            ax += sA * xA; ay += sA * yA; az += sA * zA;
            bx += sB * xB; by += sB * yB; bz += sB * zB;
        }
    }
    for (int o = t.L >> 1; o > 0; o >>= 1) {
        ax += __shfl_xor_sync(0xffffffffu, ax, o); ay += __shfl_xor_sync(0xffffffffu, ay, o); az += __shfl_xor_sync(0xffffffffu, az, o);
        bx += __shfl_xor_sync(0xffffffffu, bx, o); by += __shfl_xor_sync(0xffffffffu, by, o); bz += __shfl_xor_sync(0xffffffffu, bz, o);
    }
    aA[0] = ax; aA[1] = ay; aA[2] = az;
    aB[0] = bx; aB[1] = by; aB[2] = bz;
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

template <int CS>
__device__ __forceinline__ void bc_sync()
{
    if constexpr (CS > 1) cg::this_cluster().sync(); else __syncthreads();
}

// One group, integrated over h by the whole cluster (rank = this CTA's rank in it).  On entry S.Y,
// S.m, S.rc, S.irc of EVERY CTA hold the group; on return S.Y of every CTA holds the result.
// S0 = CTA 0's shared memory.  Returns false on step-size underflow (uniform over the cluster).
template <int MAXN, int THREADS, int CS>
__device__ __forceinline__ bool bc_integrate(BcSmem<MAXN, THREADS> &S, BcSmem<MAXN, THREADS> *S0, const int rank,
                                             const BcLane &t, double G, double m0, double h, double eps, int *nsteps)
{
    int buf = 0;
    double done = 0.0, H = h;
    bool last = false, fresh = true;
    const double eps2 = eps * eps;
    const int i = t.i;
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
    double q[3] = {1.0, 0.0, 0.0}, V[3] = {0.0, 1.0, 0.0}, acc0[3] = {0.0, 0.0, 0.0};
    while (!last) {
        double rem = h - done;
        if (fabs(H) >= fabs(rem)) { H = rem; last = true; }
        if (fresh) {                                     // new starting state: load it, force at it
            if (t.owner) {
#pragma unroll
                for (int c = 0; c < 3; ++c) { q[c] = S.Y[c][i]; V[c] = S.Y[3 + c][i]; }
                if (rank == 0) {
                    S.isq[i] = 1.0 / (q[0] * q[0] + q[1] * q[1] + q[2] * q[2]);
                    S.isv[i] = 1.0 / (V[0] * V[0] + V[1] * V[1] + V[2] * V[2]);
                }
            }
            double dummy[3];
            bc_rhs2(S, t, buf, G, m0, q, q, acc0, dummy);
            fresh = false;
        }
        // ---- my columns: Gragg's modified midpoint rule with nk substeps
#pragma unroll 1
        for (int pass = 0; pass < BS_KMAX / CS; ++pass) {
            const int col = (pass & 1) ? pass * CS + CS - 1 - rank : pass * CS + rank;
            const int nk = 2 * (col + 1);
            const double eta = H / nk;
            double qa[3], Va[3], qb[3], Vb[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                qa[c] = q[c]; Va[c] = V[c];
                qb[c] = q[c] + eta * V[c]; Vb[c] = V[c] + eta * acc0[c];
            }
            // two substeps per iteration (bc_rhs2): q_{k+1} = q_{k-1} + 2 eta V_k does not need a(q_k)
#pragma unroll 1
            for (int it = 0; it <= col; ++it) {
                double qc[3], A[3], C[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) qc[c] = qa[c] + 2.0 * eta * Vb[c];
                bc_rhs2(S, t, buf, G, m0, qb, qc, A, C);
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    double vc = Va[c] + 2.0 * eta * A[c];
                    if (it == col && t.owner) {
                        S0->tab[col][c][i] = 0.5 * (qc[c] + qb[c] + eta * vc);
                        S0->tab[col][3 + c][i] = 0.5 * (vc + Vb[c] + eta * C[c]);
                    }
                    double qd = qb[c] + 2.0 * eta * vc, vd = Vb[c] + 2.0 * eta * C[c];
                    qa[c] = qc[c]; Va[c] = vc; qb[c] = qd; Vb[c] = vd;
                }
            }
        }
        bc_sync<CS>();
        // ---- CTA 0: Aitken-Neville tableau in (H/n_k)^2, first row whose error passes
        if (rank == 0) {
            double e[BS_KMAX];
#pragma unroll
            for (int k = 0; k < BS_KMAX; ++k) e[k] = 0.0;
            // eight lanes per body, six of them take one component each
            for (int i8 = threadIdx.x >> 3; i8 < ((t.n + 3) & ~3); i8 += THREADS / 8) {
                const int c = threadIdx.x & 7;
                double d2[BS_KMAX];
#pragma unroll
                for (int k = 0; k < BS_KMAX; ++k) d2[k] = 0.0;
                if (c < 6 && i8 < t.n) {
                    double row[BS_KMAX] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
                    for (int k = 0; k < BS_KMAX; ++k) {
                        double cur = S.tab[k][c][i8], prev = row[0], diff = 0.0;
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
                        S.tab[k][c][i8] = cur;                      // T[k][k]
                        d2[k] = diff * diff;
                    }
                }
                const int base = (threadIdx.x & 31) & ~7;
                const double isq = i8 < t.n ? S.isq[i8] : 0.0, isv = i8 < t.n ? S.isv[i8] : 0.0;
#pragma unroll
                for (int k = 1; k < BS_KMAX; ++k) {
                    double dq = __shfl_sync(0xffffffffu, d2[k], base) + __shfl_sync(0xffffffffu, d2[k], base + 1) + __shfl_sync(0xffffffffu, d2[k], base + 2);
                    double dv = __shfl_sync(0xffffffffu, d2[k], base + 3) + __shfl_sync(0xffffffffu, d2[k], base + 4) + __shfl_sync(0xffffffffu, d2[k], base + 5);
                    e[k] = fmax(e[k], fmax(dq * isq, dv * isv));
                }
            }
#pragma unroll
            for (int k = 1; k < BS_KMAX; ++k)
                for (int o = 16; o > 0; o >>= 1) e[k] = fmax(e[k], __shfl_xor_sync(0xffffffffu, e[k], o));
            if ((threadIdx.x & 31) == 0) {
#pragma unroll
                for (int k = 1; k < BS_KMAX; ++k) S.wmax[threadIdx.x >> 5][k] = e[k];
            }
            __syncthreads();
            int kstar = -1;
#pragma unroll
            for (int k = BS_KMAX - 1; k >= 1; --k) {
                double r = S.wmax[0][k];
#pragma unroll
                for (int w = 1; w < THREADS / 32; ++w) r = fmax(r, S.wmax[w][k]);
                if (r <= eps2) kstar = k;
            }
            if (kstar >= 0 && t.owner) {
#pragma unroll
                for (int c = 0; c < 6; ++c) S.Y[c][i] = S.tab[kstar][c][i];
            }
            if (threadIdx.x == 0) S.kstar = kstar;
        }
        bc_sync<CS>();
        const int kstar = S0->kstar;
        if (kstar >= 0) {
            if (CS > 1 && rank != 0) {
                const int n = t.n;
                for (int b = threadIdx.x; b < 6 * n; b += THREADS) {
                    int c = b / n, k = b - c * n;
                    S.Y[c][k] = S0->Y[c][k];
                }
                __syncthreads();
            }
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
