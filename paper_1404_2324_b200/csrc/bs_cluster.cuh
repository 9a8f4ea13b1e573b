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
    double pos[2][3][MAXN];
    float pf[2][3][MAXN];           // positions rounded to FP32 for the conservative pretest
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

#ifdef GENGA_TRACE
__device__ long long g_bc_prof[1024][8];     // per CTA: cycles in rhs, cluster syncs, tableau, attempts
#define BC_T0() long long tq_ = clock64()
#define BC_ACC(k) do { long long tn_ = clock64(); if (threadIdx.x == 0) g_bc_prof[blockIdx.x][k] += tn_ - tq_; tq_ = tn_; } while (0)
#else
#define BC_T0()
#define BC_ACC(k)
#endif
// Force on body t.i at the positions q of the owners (Eq. 1 L73-74 through Eq. 8; star fixed
// at the origin, L314; every pair of the group is examined at every evaluation, L505).  The n^2
// examinations are done first in FP32 against a threshold widened by more than the FP32 rounding,
// so the test can only err towards "inside"; pairs that pass take the exact FP64 test and weight.
template <int MAXN, int THREADS>
__device__ __forceinline__ void bc_rhs(BcSmem<MAXN, THREADS> &S, const BcLane &t, int &buf, double G, double m0,
                                       const double q[3], double a[3])
{
    GENGA_BS_RHS_HOOK();
    BC_T0();
    double(*p)[MAXN] = S.pos[buf];
    float(*pf)[MAXN] = S.pf[buf];
    if (t.owner) {
        p[0][t.i] = q[0]; p[1][t.i] = q[1]; p[2][t.i] = q[2];
        pf[0][t.i] = (float)q[0]; pf[1][t.i] = (float)q[1]; pf[2][t.i] = (float)q[2];
    }
    __syncthreads();
    BC_ACC(4);
    buf ^= 1;
    double ax = 0.0, ay = 0.0, az = 0.0;
    if (t.i < t.n) {
        const int n = t.n, L = t.L, i = t.i;
        const float fx = pf[0][i], fy = pf[1][i], fz = pf[2][i], ft = S.thr2[i];
        const double qx = p[0][i], qy = p[1][i], qz = p[2][i];
        const double my_rc = S.rc[i], my_irc = S.irc[i];
        for (int j0 = t.s; j0 <= n; j0 += 32 * L) {              // partner j = n is the star
            unsigned mask = 0u;
#pragma unroll 4
            for (int kk = 0; kk < 32; ++kk) {
                int j = j0 + kk * L;
                if (j > n) break;
                int jc = j < n ? j : i;                           // star / self: computed, not used
                float dx = pf[0][jc] - fx, dy = pf[1][jc] - fy, dz = pf[2][jc] - fz;
                float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                bool in = (d2 < fmaxf(ft, S.thr2[jc]) && j != i) || j == n;
                mask |= (in ? 1u : 0u) << kk;
            }
            BC_ACC(5);
            while (mask) {
                int j = j0 + (__ffs(mask) - 1) * L;
                mask &= mask - 1;
                if (j == n) {
                    double r2 = qx * qx + qy * qy + qz * qz;
                    double s0 = -G * m0 * rinv3_fast(r2);
                    ax += s0 * qx; ay += s0 * qy; az += s0 * qz;
                } else {
                    double rcj = S.rc[j];
                    double rcij = fmax(my_rc, rcj);
                    double dx = p[0][j] - qx, dy = p[1][j] - qy, dz = p[2][j] - qz;
                    double d2 = dx * dx + dy * dy + dz * dz;
                    if (d2 < rcij * rcij) {
                        double sc = direct_scale(d2, rcij, my_rc >= rcj ? my_irc : S.irc[j], G * S.m[j]);
                        ax += sc * dx; ay += sc * dy; az += sc * dz;
                    }
                }
            }
        }
    }
    BC_ACC(6);
    for (int o = t.L >> 1; o > 0; o >>= 1) {
        ax += __shfl_xor_sync(0xffffffffu, ax, o);
        ay += __shfl_xor_sync(0xffffffffu, ay, o);
        az += __shfl_xor_sync(0xffffffffu, az, o);
    }
    a[0] = ax; a[1] = ay; a[2] = az;
    BC_ACC(7);
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
    double q[3] = {1.0, 0.0, 0.0}, V[3] = {0.0, 1.0, 0.0}, isq = 0.0, isv = 0.0, acc0[3] = {0.0, 0.0, 0.0};
    while (!last) {
        double rem = h - done;
        if (fabs(H) >= fabs(rem)) { H = rem; last = true; }
        if (fresh) {                                     // new starting state: load it, force at it
            if (t.owner) {
#pragma unroll
                for (int c = 0; c < 3; ++c) { q[c] = S.Y[c][i]; V[c] = S.Y[3 + c][i]; }
                isq = 1.0 / (q[0] * q[0] + q[1] * q[1] + q[2] * q[2]);
                isv = 1.0 / (V[0] * V[0] + V[1] * V[1] + V[2] * V[2]);
            }
            bc_rhs(S, t, buf, G, m0, q, acc0);
            fresh = false;
        }
        BC_T0();
        // ---- my columns: Gragg's modified midpoint rule with nk substeps
#pragma unroll 1
        for (int pass = 0; pass < BS_KMAX / CS; ++pass) {
            const int col = (pass & 1) ? pass * CS + CS - 1 - rank : pass * CS + rank;
            const int nk = 2 * (col + 1);
            const double eta = H / nk;
            double qa[3], Va[3], qb[3], Vb[3], acc[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                qa[c] = q[c]; Va[c] = V[c];
                qb[c] = q[c] + eta * V[c]; Vb[c] = V[c] + eta * acc0[c];
            }
#pragma unroll 1
            for (int ms = 1; ms < nk; ++ms) {
                bc_rhs(S, t, buf, G, m0, qb, acc);
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    double qn = qa[c] + 2.0 * eta * Vb[c];
                    double vn = Va[c] + 2.0 * eta * acc[c];
                    qa[c] = qb[c]; Va[c] = Vb[c]; qb[c] = qn; Vb[c] = vn;
                }
            }
            bc_rhs(S, t, buf, G, m0, qb, acc);
            if (t.owner) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    S0->tab[col][c][i] = 0.5 * (qb[c] + qa[c] + eta * Vb[c]);
                    S0->tab[col][3 + c][i] = 0.5 * (Vb[c] + Va[c] + eta * acc[c]);
                }
            }
        }
        BC_ACC(0);
        bc_sync<CS>();
        BC_ACC(1);
        // ---- CTA 0: Aitken-Neville tableau in (H/n_k)^2, first row whose error passes
        if (rank == 0) {
            double e[BS_KMAX];
#pragma unroll
            for (int k = 0; k < BS_KMAX; ++k) e[k] = 0.0;
            if (t.owner) {
                double dq2[BS_KMAX], dv2[BS_KMAX];
#pragma unroll
                for (int k = 0; k < BS_KMAX; ++k) { dq2[k] = 0.0; dv2[k] = 0.0; }
#pragma unroll
                for (int c = 0; c < 6; ++c) {
                    double row[BS_KMAX] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
                    for (int k = 0; k < BS_KMAX; ++k) {
                        double cur = S.tab[k][c][i], prev = row[0], diff = 0.0;
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
                        S.tab[k][c][i] = cur;                       // T[k][k]
                        if (c < 3) dq2[k] += diff * diff; else dv2[k] += diff * diff;
                    }
                }
#pragma unroll
                for (int k = 1; k < BS_KMAX; ++k) e[k] = fmax(dq2[k] * isq, dv2[k] * isv);
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
        BC_ACC(2);
        bc_sync<CS>();
        BC_ACC(1);
#ifdef GENGA_TRACE
        if (threadIdx.x == 0) g_bc_prof[blockIdx.x][3] += 1;
#endif
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
