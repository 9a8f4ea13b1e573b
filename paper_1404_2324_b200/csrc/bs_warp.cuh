// Force evaluation of Bulirsch-Stoer for one SMALL close-encounter group (2..8 bodies; the
// paper's Table 3, gives groups of 2 a block of 4 threads), used by the block layout of bs_small.cuh.
//
// Most groups are pairs and triples (cfg1: 140 of 165 groups; cfg2, cfg3, cfg4: nearly all), and what a group costs is the
// LENGTH of its dependent chain.  The modified-midpoint runs (n_k = 2, 4, ..., 16 substeps, all from the same state) sit
// side by side in the lanes of a warp, S = 2, 4 or 8 lanes per column segment, one lane per body; a lane keeps its body's
// midpoint state in registers.  S = 2, 4: the positions of the other bodies of the SAME column come by segmented
// shuffles (no shared memory, no barrier on the chain; every partner slot is evaluated, without a branch: these
// evaluations are bound by FP64 issue, a shared-memory exchange measured the same).  S = 8: see bw_rhs2_seg8.
#pragma once
#include "bs.cuh"

namespace genga {

constexpr int BW_MAXN = 8;          // largest group of the warp layout
constexpr int BW_WARPS = 4;         // warps per block: one per SM sub-partition

// Forces on this lane's body at TWO positions qA, qB at once; the partners are the other lanes of its
// S-lane segment (same column): partner t = 0..n-2 sits in segment lane src[t] = (b + 1 + t) mod n and
// carries rcij[t] = max(rc_b, rc_j) (0 for a massless or missing partner, so that it never passes the
// test), irc[t] = 1 / (0.9 rcij), gm[t] = G m_j.  Star fixed at the origin (L314); every pair of the group
// is examined at every evaluation (L505).
// Why two: in Gragg's rule q_{k+1} = q_{k-1} + 2 eta V_k and V_{k+1} = V_{k-1} + 2 eta a(q_k), so a(q_k)
// and a(q_{k+1}) do not depend on each other; evaluated in one straight-line block their two dependent
// chains (~300 cycles each: shuffle, distance, changeover weight) overlap.  No branch on the data (a partner
// outside rc_ij is computed and discarded).
template <int S>
__device__ __forceinline__ void bw_rhs2(const double (&qA)[3], const double (&qB)[3], double Gm0, const int (&src)[S],
                                        const double (&rcij)[S], const double (&irc)[S], const double (&gm)[S],
                                        const int n, double (&aA)[3], double (&aB)[3])
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
        if (t < n - 1) {                                          // a triple in four lanes: its third partner slot is empty (uniform)
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
// weight is evaluated once per close pair instead of once per partner slot: (1) an FP32 pretest of the n - 1
// partners at both points against a threshold widened by more than the FP32 rounding (it can only err towards
// "inside"), one bit per partner that may be inside rc_ij at either point; (2) while any lane has a bit left, every
// lane takes ITS next close partner, makes the exact FP64 test, evaluates both weights and accumulates.  Rounds = the
// largest number of close partners of any body (typically 1 or 2).
// Positions go through shared memory (the segment's slot: one STS.128 per two doubles, one LDS.128 per two doubles of
// a partner) instead of shuffles: a 64-bit shuffle costs 8.7 issue cycles of the warp's scheduler against 2.1 for a
// DFMA (measured, B200), and phase 1 alone was 84 of them (150 cycles per partner; 40 % of an evaluation).
struct BwSlot8 {
    double2 q[8][3];          // body: (Ax, Ay), (Az, Bx), (By, Bz)
    float4 f[2][8];           // the two points rounded to FP32, .w = the body's pretest threshold (rc + margin)^2
};
struct BwGroup8 {
    double2 rcm[8];           // (rc_j, G m_j) of the group's bodies
};

__device__ __forceinline__ void bw_rhs2_seg8(const BwGroup8 &W, BwSlot8 &P, const double (&qA)[3], const double (&qB)[3], const int n, const int b,
                                             double Gm0, double my_rc, const float thr, const unsigned massive,
                                             double (&aA)[3], double (&aB)[3])
{
    GENGA_BS_RHS_HOOK();
    const unsigned full = 0xffffffffu;
    __syncwarp();                                                 // the slot's previous contents have been read
    const float fAx = (float)qA[0], fAy = (float)qA[1], fAz = (float)qA[2], fBx = (float)qB[0], fBy = (float)qB[1], fBz = (float)qB[2];
    P.q[b][0] = make_double2(qA[0], qA[1]); P.q[b][1] = make_double2(qA[2], qB[0]); P.q[b][2] = make_double2(qB[1], qB[2]);
    P.f[0][b] = make_float4(fAx, fAy, fAz, thr);
    P.f[1][b] = make_float4(fBx, fBy, fBz, thr);
    double rA = fma(qA[2], qA[2], fma(qA[1], qA[1], qA[0] * qA[0]));
    double rB = fma(qB[2], qB[2], fma(qB[1], qB[1], qB[0] * qB[0]));
    double sA = -Gm0 * rinv3_fast(rA), sB = -Gm0 * rinv3_fast(rB);
    double ax = sA * qA[0], ay = sA * qA[1], az = sA * qA[2];
    double bx = sB * qB[0], by = sB * qB[1], bz = sB * qB[2];
    __syncwarp();
    // (1) bit j: body j (massive, not this one) may be inside max(rc_b, rc_j) at A or B
    unsigned close = 0u;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        const float4 pa = P.f[0][j], pb = P.f[1][j];
        const float dx = pa.x - fAx, dy = pa.y - fAy, dz = pa.z - fAz, ex = pb.x - fBx, ey = pb.y - fBy, ez = pb.z - fBz;
        const float d2 = fminf(fmaf(dz, dz, fmaf(dy, dy, dx * dx)), fmaf(ez, ez, fmaf(ey, ey, ex * ex)));
        close |= d2 < fmaxf(thr, pa.w) ? 1u << j : 0u;
    }
    close &= massive & ~(1u << b);
    close = b < n ? close : 0u;
    // (2)
    while (__any_sync(full, close != 0u)) {
        const bool act = close != 0u;
        const int j = act ? __ffs(close) - 1 : b;
        close &= close - 1;
        const double2 p0 = P.q[j][0], p1 = P.q[j][1], p2 = P.q[j][2], rm = W.rcm[j];
        const double dxA = p0.x - qA[0], dyA = p0.y - qA[1], dzA = p1.x - qA[2];
        const double dxB = p1.y - qB[0], dyB = p2.x - qB[1], dzB = p2.y - qB[2];
        const double r = my_rc >= rm.x ? my_rc : rm.x, rc2 = r * r;
        const double dA = fma(dzA, dzA, fma(dyA, dyA, dxA * dxA)), dB = fma(dzB, dzB, fma(dyB, dyB, dxB * dxB));
        const bool inA = act && dA < rc2, inB = act && dB < rc2;
        const double ir = rcp_fast(0.9 * (act ? r : 1.0));
        double scA = direct_scale_nb(inA ? dA : 1.0, r, ir, rm.y), scB = direct_scale_nb(inB ? dB : 1.0, r, ir, rm.y);
        scA = inA ? scA : 0.0; scB = inB ? scB : 0.0;
        ax = fma(scA, dxA, ax); ay = fma(scA, dyA, ay); az = fma(scA, dzA, az);
        bx = fma(scB, dxB, bx); by = fma(scB, dyB, by); bz = fma(scB, dzB, bz);
    }
    aA[0] = ax; aA[1] = ay; aA[2] = az;
    aB[0] = bx; aB[1] = by; aB[2] = bz;
}

}  // namespace genga
