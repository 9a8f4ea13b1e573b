// Bulirsch-Stoer integration of H_A for one close-encounter group (
// Eq. 1).  The star is fixed at the origin during the step (L314); every pair of
// the group interacts, indirect ones included (L505), with the weight 1 - W of the part
// of the pair force that the changeover function moved from H_B to H_A.
//
// Algorithm: Gragg's modified midpoint rule with the substep
// sequence n_k = 2,4,...,16, Aitken-Neville extrapolation in (H/n_k)^2, relative error
// max_i max(|dq_i|^2/|q_i|^2, |dV_i|^2/|V_i|^2) between the last two entries of a tableau
// row, accept at <= eps^2; on failure after 8 columns H <- H/2, after an accept within five
// columns H <- 1.5 H, the last step is cut to land exactly on h.
//
// Two layouts in this file (the paper's Table 3, picked block sizes for cc 2.x; the warp and
// cluster layouts are in bs_warp.cuh and bs_cluster.cuh):
//   * team of TW lanes of one warp, one body per lane, everything in registers, positions
//     exchanged through double-buffered shared memory (one __syncwarp per force evaluation);
//   * one thread block per large group, bodies strided over the threads, tableau in a
//     global scratch area (any group size, up to all 2048 bodies, Fig. 15).
// Every integrator counts into nsteps[2]: [0] accepted steps, [1] rejected attempts (all 8 columns failed).
#pragma once
#include "common.cuh"

#ifndef GENGA_BS_RHS_HOOK
#define GENGA_BS_RHS_HOOK()          // profiling builds count force evaluations here
#endif

namespace genga {

constexpr int BS_KMAX = 8;
constexpr double BS_HMIN = 1e-12;

// 1 / ((n_k / n_{k-j})^2 - 1) of the Aitken-Neville recurrence for n_k = 2(k+1)
struct BsIden { double v[BS_KMAX][BS_KMAX]; };
constexpr BsIden bs_make_iden()
{
    BsIden t{};
    for (int k = 0; k < BS_KMAX; ++k)
        for (int j = 1; j <= k; ++j) {
            double r = double(k + 1) / double(k - j + 1);
            t.v[k][j] = 1.0 / (r * r - 1.0);
        }
    return t;
}
static __constant__ BsIden c_bs_iden = bs_make_iden();

template <int TW>
struct WarpTeam {
    unsigned mask;
    int lane;  // 0..TW-1 inside the team
    __device__ __forceinline__ void sync() const { __syncwarp(mask); }
    __device__ __forceinline__ double max(double v) const
    {
#pragma unroll
        for (int o = TW / 2; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(mask, v, o, TW));
        return v;
    }
};

// shared memory of one team: masses, critical radii, two position buffers
template <int TW>
struct TeamSmem {
    double m[TW], rc[TW], irc[TW];      // irc = 1 / (0.9 rc)
    double p[2][3][TW];
};

// acceleration of the team's body `lane` at positions q (of all team bodies)
template <int TW>
__device__ __forceinline__ void bs_rhs(const WarpTeam<TW> &t, TeamSmem<TW> &sm, int &buf, int nb,
                                       unsigned srcmask, double G, double m0, double my_rc,
                                       const double q[3], double a[3])
{
    GENGA_BS_RHS_HOOK();
    double(*p)[TW] = sm.p[buf];
    p[0][t.lane] = q[0]; p[1][t.lane] = q[1]; p[2][t.lane] = q[2];
    t.sync();
    buf ^= 1;
    double r2 = q[0] * q[0] + q[1] * q[1] + q[2] * q[2];
    double s0 = -G * m0 * rinv3_fast(r2);
    double ax = s0 * q[0], ay = s0 * q[1], az = s0 * q[2];
    const double my_irc = sm.irc[t.lane];
    for (int j = 0; j < nb; ++j) {
        if (j == t.lane || !((srcmask >> j) & 1u)) continue;
        double mj = sm.m[j];
        if (mj == 0.0) continue;
        double rcj = sm.rc[j];
        double rcij = fmax(my_rc, rcj);
        double dx = p[0][j] - q[0], dy = p[1][j] - q[1], dz = p[2][j] - q[2];
        double d2 = dx * dx + dy * dy + dz * dz;
        if (d2 < rcij * rcij) {
            double s = direct_scale(d2, rcij, my_rc >= rcj ? my_irc : sm.irc[j], G * mj);
            ax += s * dx; ay += s * dy; az += s * dz;
        }
    }
    a[0] = ax; a[1] = ay; a[2] = az;
}

// Integrate the team's bodies over h.  q, V in registers (in/out).  `active` lanes own a
// body; srcmask marks the slots that exist (bit j = slot j).  Returns false on step underflow.
template <int TW>
__device__ bool bs_team(const WarpTeam<TW> &t, TeamSmem<TW> &sm, int nb, bool active, unsigned srcmask,
                        double G, double m0, double my_rc, double q[3], double V[3], double h,
                        double eps, int *nsteps)
{
    int buf = 0;
    double done = 0.0, H = h;
    bool last = false;
    const double eps2 = eps * eps;
    double row[BS_KMAX][6];
    while (!last) {
        double rem = h - done;
        if (fabs(H) >= fabs(rem)) { H = rem; last = true; }
        double sq = q[0] * q[0] + q[1] * q[1] + q[2] * q[2];
        double sv = V[0] * V[0] + V[1] * V[1] + V[2] * V[2];
        double isq = active ? 1.0 / sq : 0.0, isv = active ? 1.0 / sv : 0.0;
        double acc0[3];
        bs_rhs<TW>(t, sm, buf, nb, srcmask, G, m0, my_rc, q, acc0);
        bool accepted = false;
        while (!accepted) {
#pragma unroll
            for (int k = 0; k < BS_KMAX; ++k) {
                if (accepted) break;
                const int nk = 2 * (k + 1);
                const double eta = H / nk;
                double qa[3], Va[3], qb[3], Vb[3], acc[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    qa[c] = q[c]; Va[c] = V[c];
                    qb[c] = q[c] + eta * V[c]; Vb[c] = V[c] + eta * acc0[c];
                }
#pragma unroll 1
                for (int ms = 1; ms < nk; ++ms) {
                    bs_rhs<TW>(t, sm, buf, nb, srcmask, G, m0, my_rc, qb, acc);
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        double qn = qa[c] + 2.0 * eta * Vb[c];
                        double vn = Va[c] + 2.0 * eta * acc[c];
                        qa[c] = qb[c]; Va[c] = Vb[c]; qb[c] = qn; Vb[c] = vn;
                    }
                }
                bs_rhs<TW>(t, sm, buf, nb, srcmask, G, m0, my_rc, qb, acc);
                double T[6], prev[6];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    T[c] = 0.5 * (qb[c] + qa[c] + eta * Vb[c]);
                    T[3 + c] = 0.5 * (Vb[c] + Va[c] + eta * acc[c]);
                }
#pragma unroll
                for (int c = 0; c < 6; ++c) { prev[c] = row[0][c]; row[0][c] = T[c]; }
#pragma unroll
                for (int j = 1; j <= k; ++j) {
                    const double ratio = double(k + 1) / double(k - j + 1);
                    const double iden = 1.0 / (ratio * ratio - 1.0);
#pragma unroll
                    for (int c = 0; c < 6; ++c) {
                        double tmp = row[j][c];
                        row[j][c] = row[j - 1][c] + (row[j - 1][c] - prev[c]) * iden;
                        prev[c] = tmp;
                    }
                }
                if (k >= 1) {
                    double dq2 = 0.0, dv2 = 0.0;
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        double dq = row[k][c] - row[k - 1][c], dv = row[k][3 + c] - row[k - 1][3 + c];
                        dq2 += dq * dq; dv2 += dv * dv;
                    }
                    double e = t.max(fmax(dq2 * isq, dv2 * isv));
                    if (e <= eps2) {
#pragma unroll
                        for (int c = 0; c < 3; ++c) { q[c] = row[k][c]; V[c] = row[k][3 + c]; }
                        done += H;
                        if (nsteps) ++nsteps[0];
                        if (k <= 4) H *= 1.5;
                        accepted = true;
                    }
                }
            }
            if (!accepted) {
                H *= 0.5; last = false;
                if (nsteps) ++nsteps[1];
                if (fabs(H) < BS_HMIN * fabs(h)) return false;
            }
        }
    }
    return true;
}

// ---------------------------------------------------------------------------------
// Block layout for groups larger than a warp.  Scratch: 71 arrays of `stride` doubles; the
// group uses entries [off, off+nb).  idx[b] = global body index of member b.
struct BsScratch {
    double *base;
    int64_t stride;
    __device__ __forceinline__ double *arr(int k) const { return base + (int64_t)k * stride; }
};
enum : int { BSA_Y = 0, BSA_QA = 6, BSA_VA = 9, BSA_QB = 12, BSA_VB = 15, BSA_ACC0 = 18,
             BSA_ACC = 21, BSA_ISQ = 24, BSA_ISV = 25, BSA_M = 26, BSA_RC = 27, BSA_ROW = 28,
             BSA_COUNT = 28 + 6 * BS_KMAX,
             // the layout with collisions (k_bs_generic) carries radius, kind (0 massive, 1 test particle, 2 removed), spin
             // and the member's index within its system as well
             BSA_R = BSA_COUNT, BSA_KIND = BSA_COUNT + 1, BSA_SPIN = BSA_COUNT + 2, BSA_GIDX = BSA_COUNT + 5,
             BSA_COUNT2 = BSA_COUNT + 6 };

// ---------------------------------------------------------------------------------
// Collisions (section 3.2.7; readings R-19..R-21).  "To find collisions between the
// Bulirsch-Stoer time steps, we use the same code as in the close encounter detection" (L328): after every accepted
// Bulirsch-Stoer step the minimum of the cubic Hermite interpolant of the squared separation over that step (Eq. 10-12)
// is compared, pair by pair, with (R_i + R_j)^2.
constexpr int GENGA_EV = 24;        // doubles per event record (include/genga.h)

// a cheap lower bound of the Hermite interpolant first: P(t) = h00 P0 + h01 P1 + h10 h Pd0 + h11 h Pd1 with
// h00 + h01 = 1 and |h10|, |h11| <= 4/27 on [0, 1]
__device__ __forceinline__ bool pair_collides(double P0, double P1, double Pd0, double Pd1, double H, double Rs)
{
    const double Rs2 = Rs * Rs;
    if (fmin(P0, P1) - (4.0 / 27.0) * (fabs(H * Pd0) + fabs(H * Pd1)) > Rs2) return false;
    return hermite_min(P0, P1, Pd0, Pd1, H) < Rs2;
}

struct BsColl {
    double *ev;                     // event records, GENGA_EV doubles each
    long long evcap;
    unsigned long long *nev;        // events so far (device counter)
    double *U;                      // internal energy of this system (L318-322)
    double step_id;
    int base;                       // global index of the system's first body
    int record_massive;             // 0: a test particle's group re-enacts the massive bodies' collisions silently (L342)
};

// The merges of one accepted step, in the order of the member list (a < b), a body removed earlier in the step
// skipped: ONE thread, exactly the oracle's loop.  Old state in BSA_Y, new state in BSA_ROW + 6 k.
__device__ inline void bs_collisions_seq(const BsScratch &S, int off, int nb, int k, double H, double G, double m0, const BsColl &cc)
{
    double *m = S.arr(BSA_M) + off, *R = S.arr(BSA_R) + off, *kind = S.arr(BSA_KIND) + off, *gidx = S.arr(BSA_GIDX) + off;
    double *q0[3], *V0[3], *q1[3], *V1[3], *sp[3];
    for (int c = 0; c < 3; ++c) {
        q0[c] = S.arr(BSA_Y + c) + off; V0[c] = S.arr(BSA_Y + 3 + c) + off;
        q1[c] = S.arr(BSA_ROW + 6 * k + c) + off; V1[c] = S.arr(BSA_ROW + 6 * k + 3 + c) + off;
        sp[c] = S.arr(BSA_SPIN + c) + off;
    }
    for (int a = 0; a < nb; ++a)
        for (int b = a + 1; b < nb; ++b) {
            if (kind[a] == 2.0 || kind[b] == 2.0) continue;
            if (kind[a] == 1.0 && kind[b] == 1.0) continue;
            double d0[3], w0[3], d1[3], w1[3];
            for (int c = 0; c < 3; ++c) {
                d0[c] = q0[c][b] - q0[c][a]; w0[c] = V0[c][b] - V0[c][a];
                d1[c] = q1[c][b] - q1[c][a]; w1[c] = V1[c][b] - V1[c][a];
            }
            const double P0 = d0[0] * d0[0] + d0[1] * d0[1] + d0[2] * d0[2], Pd0 = 2.0 * (d0[0] * w0[0] + d0[1] * w0[1] + d0[2] * w0[2]);
            const double P1 = d1[0] * d1[0] + d1[1] * d1[1] + d1[2] * d1[2], Pd1 = 2.0 * (d1[0] * w1[0] + d1[1] * w1[1] + d1[2] * w1[2]);
            if (!pair_collides(P0, P1, Pd0, Pd1, H, R[a] + R[b])) continue;
            int sv = a, dd = b, kev = 0;
            if (kind[a] == 1.0) { sv = b; dd = a; kev = 1; }
            else if (kind[b] == 1.0) { sv = a; dd = b; kev = 1; }
            else if (m[b] > m[a]) { sv = b; dd = a; }
            const double ma = m[sv], mb = m[dd], mt = ma + mb;
            const bool rec = kev == 1 || cc.record_massive;
            double *e = nullptr;
            if (rec) {
                const unsigned long long slot = atomicAdd(cc.nev, 1ull);
                if ((long long)slot < cc.evcap) {
                    e = cc.ev + GENGA_EV * slot;
                    e[0] = cc.step_id; e[1] = kev; e[2] = cc.base + gidx[sv]; e[3] = cc.base + gidx[dd];
                    e[4] = ma; e[5] = mb; e[6] = R[sv]; e[7] = R[dd];
                    for (int c = 0; c < 3; ++c) { e[8 + c] = q0[c][sv]; e[11 + c] = V0[c][sv]; e[14 + c] = q0[c][dd]; e[17 + c] = V0[c][dd]; }
                }
            }
            double Uev = 0.0;
            if (kev == 0) {
                double dq[3], dv[3], r2 = 0.0, v2 = 0.0;
                for (int c = 0; c < 3; ++c) {
                    dq[c] = q1[c][sv] - q1[c][dd]; dv[c] = V1[c][sv] - V1[c][dd];
                    r2 += dq[c] * dq[c]; v2 += dv[c] * dv[c];
                }
                const double mu = ma * mb / mt;
                Uev = 0.5 * mu * v2 - G * ma * mb / sqrt(r2);
                if (cc.record_massive) atomicAdd(cc.U, Uev);
                sp[0][sv] += sp[0][dd] + mu * (dq[1] * dv[2] - dq[2] * dv[1]);
                sp[1][sv] += sp[1][dd] + mu * (dq[2] * dv[0] - dq[0] * dv[2]);
                sp[2][sv] += sp[2][dd] + mu * (dq[0] * dv[1] - dq[1] * dv[0]);
                for (int c = 0; c < 3; ++c) {
                    q1[c][sv] = (ma * q1[c][sv] + mb * q1[c][dd]) / mt;
                    V1[c][sv] = (ma * V1[c][sv] + mb * V1[c][dd]) / mt;
                }
                R[sv] = cbrt(R[sv] * R[sv] * R[sv] + R[dd] * R[dd] * R[dd]);
                m[sv] = mt;
            }
            if (e) { e[20] = Uev; e[21] = sp[0][sv]; e[22] = sp[1][sv]; e[23] = sp[2][sv]; }
            // the ghost: massless, parked far away on a circular orbit (it meets nothing and adds exact zeros to every sum)
            const double Rp = 1000.0 * (gidx[dd] + 1.0);
            m[dd] = 0.0; R[dd] = 0.0; kind[dd] = 2.0;
            sp[0][dd] = sp[1][dd] = sp[2][dd] = 0.0;
            q1[0][dd] = Rp; q1[1][dd] = 0.0; q1[2][dd] = 0.0;
            V1[0][dd] = 0.0; V1[1][dd] = sqrt(G * m0 / Rp); V1[2][dd] = 0.0;
        }
}

// Does any pair of the group collide in the step just accepted (old state BSA_Y, new state BSA_ROW + 6 k)?  All
// threads of the block; the same answer in every thread.
__device__ inline bool bs_any_collision(const BsScratch &S, int off, int nb, int k, double H)
{
    const double *R = S.arr(BSA_R) + off, *kind = S.arr(BSA_KIND) + off;
    int hit = 0;
    for (int a = threadIdx.x; a < nb && !hit; a += blockDim.x) {
        if (kind[a] == 2.0) continue;
        double qa0[3], va0[3], qa1[3], va1[3];
        for (int c = 0; c < 3; ++c) {
            qa0[c] = S.arr(BSA_Y + c)[off + a]; va0[c] = S.arr(BSA_Y + 3 + c)[off + a];
            qa1[c] = S.arr(BSA_ROW + 6 * k + c)[off + a]; va1[c] = S.arr(BSA_ROW + 6 * k + 3 + c)[off + a];
        }
        for (int b = a + 1; b < nb; ++b) {
            if (kind[b] == 2.0 || (kind[a] == 1.0 && kind[b] == 1.0)) continue;
            double P0 = 0.0, Pd0 = 0.0, P1 = 0.0, Pd1 = 0.0;
            for (int c = 0; c < 3; ++c) {
                const double d0 = S.arr(BSA_Y + c)[off + b] - qa0[c], w0 = S.arr(BSA_Y + 3 + c)[off + b] - va0[c];
                const double d1 = S.arr(BSA_ROW + 6 * k + c)[off + b] - qa1[c], w1 = S.arr(BSA_ROW + 6 * k + 3 + c)[off + b] - va1[c];
                P0 += d0 * d0; Pd0 += 2.0 * d0 * w0; P1 += d1 * d1; Pd1 += 2.0 * d1 * w1;
            }
            if (pair_collides(P0, P1, Pd0, Pd1, H, R[a] + R[b])) { hit = 1; break; }
        }
    }
    return __syncthreads_or(hit) != 0;
}

__device__ inline void bsb_rhs(const BsScratch &S, int off, int nb, double G, double m0, int posarr, int accarr)
{
    const double *px = S.arr(posarr) + off, *py = S.arr(posarr + 1) + off, *pz = S.arr(posarr + 2) + off;
    const double *pm = S.arr(BSA_M) + off, *prc = S.arr(BSA_RC) + off;
    for (int b = threadIdx.x; b < nb; b += blockDim.x) {
        double qx = px[b], qy = py[b], qz = pz[b], my_rc = prc[b];
        double r2 = qx * qx + qy * qy + qz * qz, r = sqrt(r2);
        double s0 = -G * m0 / (r2 * r);
        double ax = s0 * qx, ay = s0 * qy, az = s0 * qz;
        for (int j = 0; j < nb; ++j) {
            if (j == b) continue;
            double mj = pm[j];
            if (mj == 0.0) continue;
            double rcij = fmax(my_rc, prc[j]);
            double dx = px[j] - qx, dy = py[j] - qy, dz = pz[j] - qz;
            double d2 = dx * dx + dy * dy + dz * dz;
            if (d2 < rcij * rcij) {
                double d = sqrt(d2);
                double w = 1.0 - kick_weight(d, rcij);
                double s = G * mj / (d2 * d) * w;
                ax += s * dx; ay += s * dy; az += s * dz;
            }
        }
        S.arr(accarr)[off + b] = ax; S.arr(accarr + 1)[off + b] = ay; S.arr(accarr + 2)[off + b] = az;
    }
    __syncthreads();
}

// red: shared double[32]
__device__ inline double block_max(double v, double *red)
{
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    int nw = (blockDim.x + 31) >> 5;
    double r = red[0];
    for (int w = 1; w < nw; ++w) r = fmax(r, red[w]);
    return r;
}

// state Y (arrays BSA_Y..+5), m, rc must be loaded at [off, off+nb) before the call.
__device__ inline bool bs_block(const BsScratch &S, int off, int nb, double G, double m0, double h,
                                double eps, double *red, int *nsteps, const BsColl *cc = nullptr)
{
    double done = 0.0, H = h;
    bool last = false;
    const double eps2 = eps * eps;
    __syncthreads();
    while (!last) {
        double rem = h - done;
        if (fabs(H) >= fabs(rem)) { H = rem; last = true; }
        for (int b = threadIdx.x; b < nb; b += blockDim.x) {
            double sq = 0, sv = 0;
            for (int c = 0; c < 3; ++c) {
                double a = S.arr(BSA_Y + c)[off + b], v = S.arr(BSA_Y + 3 + c)[off + b];
                sq += a * a; sv += v * v;
            }
            S.arr(BSA_ISQ)[off + b] = 1.0 / sq; S.arr(BSA_ISV)[off + b] = 1.0 / sv;
        }
        bsb_rhs(S, off, nb, G, m0, BSA_Y, BSA_ACC0);
        bool accepted = false;
        while (!accepted) {
            for (int k = 0; k < BS_KMAX && !accepted; ++k) {
                const int nk = 2 * (k + 1);
                const double eta = H / nk;
                for (int b = threadIdx.x; b < nb; b += blockDim.x)
                    for (int c = 0; c < 3; ++c) {
                        double q = S.arr(BSA_Y + c)[off + b], v = S.arr(BSA_Y + 3 + c)[off + b];
                        S.arr(BSA_QA + c)[off + b] = q; S.arr(BSA_VA + c)[off + b] = v;
                        S.arr(BSA_QB + c)[off + b] = q + eta * v;
                        S.arr(BSA_VB + c)[off + b] = v + eta * S.arr(BSA_ACC0 + c)[off + b];
                    }
                __syncthreads();
                for (int ms = 1; ms < nk; ++ms) {
                    bsb_rhs(S, off, nb, G, m0, BSA_QB, BSA_ACC);
                    for (int b = threadIdx.x; b < nb; b += blockDim.x)
                        for (int c = 0; c < 3; ++c) {
                            double qa = S.arr(BSA_QA + c)[off + b], va = S.arr(BSA_VA + c)[off + b];
                            double qb = S.arr(BSA_QB + c)[off + b], vb = S.arr(BSA_VB + c)[off + b];
                            double qn = qa + 2.0 * eta * vb;
                            double vn = va + 2.0 * eta * S.arr(BSA_ACC + c)[off + b];
                            S.arr(BSA_QA + c)[off + b] = qb; S.arr(BSA_VA + c)[off + b] = vb;
                            S.arr(BSA_QB + c)[off + b] = qn; S.arr(BSA_VB + c)[off + b] = vn;
                        }
                    __syncthreads();
                }
                bsb_rhs(S, off, nb, G, m0, BSA_QB, BSA_ACC);
                double e = 0.0;
                for (int b = threadIdx.x; b < nb; b += blockDim.x) {
                    double dq2 = 0.0, dv2 = 0.0;
                    for (int c = 0; c < 6; ++c) {
                        double qa = S.arr(c < 3 ? BSA_QA + c : BSA_VA + c - 3)[off + b];
                        double qb = S.arr(c < 3 ? BSA_QB + c : BSA_VB + c - 3)[off + b];
                        double der = c < 3 ? S.arr(BSA_VB + c)[off + b] : S.arr(BSA_ACC + c - 3)[off + b];
                        double T = 0.5 * (qb + qa + eta * der);
                        double prev = S.arr(BSA_ROW + c)[off + b];
                        S.arr(BSA_ROW + c)[off + b] = T;
                        double cur = T, diff = 0.0;
                        for (int j = 1; j <= k; ++j) {
                            double ratio = double(k + 1) / double(k - j + 1);
                            double iden = 1.0 / (ratio * ratio - 1.0);
                            double tmp = S.arr(BSA_ROW + 6 * j + c)[off + b];
                            diff = (cur - prev) * iden;
                            cur = cur + diff;
                            S.arr(BSA_ROW + 6 * j + c)[off + b] = cur;
                            prev = tmp;
                        }
                        if (c < 3) dq2 += diff * diff; else dv2 += diff * diff;
                    }
                    e = fmax(e, fmax(dq2 * S.arr(BSA_ISQ)[off + b], dv2 * S.arr(BSA_ISV)[off + b]));
                }
                if (k >= 1) {
                    e = block_max(e, red);
                    if (e <= eps2) {
                        if (cc) {                    // collisions between the Bulirsch-Stoer steps (L328): may merge bodies in row k
                            __syncthreads();
                            if (bs_any_collision(S, off, nb, k, H)) {
                                if (threadIdx.x == 0) bs_collisions_seq(S, off, nb, k, H, G, m0, *cc);
                                __syncthreads();
                            }
                        }
                        for (int b = threadIdx.x; b < nb; b += blockDim.x)
                            for (int c = 0; c < 6; ++c) S.arr(BSA_Y + c)[off + b] = S.arr(BSA_ROW + 6 * k + c)[off + b];
                        done += H;
                        if (nsteps && threadIdx.x == 0) ++nsteps[0];
                        if (k <= 4) H *= 1.5;
                        accepted = true;
                    }
                }
                __syncthreads();
            }
            if (!accepted) {
                if (nsteps && threadIdx.x == 0) ++nsteps[1];
                H *= 0.5; last = false;
                if (fabs(H) < BS_HMIN * fabs(h)) return false;
            }
        }
    }
    return true;
}

}  // namespace genga
