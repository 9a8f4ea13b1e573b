/*
 * genga_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded FP64 CPU restatement of the hybrid symplectic
 * integrator of Grimm & Stadel, "The GENGA code".  It exists only so
 * that tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg can check
 * and time the CUDA path against it.  It shares no code with the CUDA path and
 * nothing in paper_1404_2324_b200/ may import, link or call it.
 *
 * Every function cites the passage of PAPER.md it follows.  Where the paper is
 * silent or garbled the reading taken is the one listed in DESIGN.md
 * ("Readings"), quoted here as [R-n].
 *
 * Layout: all vectors are SoA, v[c*n + i], c = 0,1,2 (x,y,z), i = body index.
 * Bodies 0..n_massive-1 are massive, n_massive..n-1 are massless test particles
 * (PAPER.md L334-342).  The star (index "0" of the paper, mass m0) sits at the
 * origin of the democratic coordinates: q = heliocentric position,
 * V = barycentric velocity.
 *
 * Parity pins: tests/test_oracle_*.py.  Unpinned readings:
 *   - ora_rcrit: the definitions of v_i and R_H,i in Eq. 6 [R-5]  -> "parity unpinned"
 *   - when r_crit is recomputed inside a higher-order step [R-4]   -> "parity unpinned"
 *   - test-particle group composition [R-12]                       -> "parity unpinned"
 *   - the Bulirsch-Stoer step-size controller [R-7] (any controller that meets
 *     the tolerance is correct; the result is pinned, the rule is not)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORA_OK        0
#define ORA_EINVAL   -1
#define ORA_ECAPACITY -2
#define ORA_EKEPLER  -3
#define ORA_EBS      -4

/* ------------------------------------------------------------------------- */
/* Compensated (Neumaier) accumulation, so the oracle's own rounding is ~1 ulp */
typedef struct { double s, c; } nsum;
static void ns_add(nsum *a, double x)
{
    double t = a->s + x;
    if (fabs(a->s) >= fabs(x)) a->c += (a->s - t) + x;
    else                       a->c += (x - t) + a->s;
    a->s = t;
}
static double ns_val(const nsum *a) { return a->s + a->c; }

/* ------------------------------------------------------------------------- */
/* Changeover function, Eq. 4-5:
 *   y = (r - 0.1 rc)/(0.9 rc);  K = 0 (y<0), y^2/(2y^2-2y+1) (0<y<1), 1 (y>1).
 * dK/dr follows by differentiating Eq. 4: dK/dy = 2y(1-y)/(2y^2-2y+1)^2,
 * dy/dr = 1/(0.9 rc).  K and dK/dr are continuous at y=0 and y=1, so the open
 * inequalities of Eq. 4 leave nothing undefined. */
void ora_changeover(double r, double rc, double *K, double *dKdr)
{
    if (rc <= 0.0) { *K = 1.0; *dKdr = 0.0; return; }
    double y = (r - 0.1 * rc) / (0.9 * rc);
    if (y <= 0.0) { *K = 0.0; *dKdr = 0.0; return; }
    if (y >= 1.0) { *K = 1.0; *dKdr = 0.0; return; }
    double D = 2.0 * y * y - 2.0 * y + 1.0;
    *K = y * y / D;
    *dKdr = 2.0 * y * (1.0 - y) / (D * D) / (0.9 * rc);
}

/* Weight of the Newtonian pair force in the kick operator B [R-1]:
 * H_B = -sum G m_i m_j K(r)/r (Eq. 2) and the operators are Hamilton's
 * equations of each part (Eq. 8), so the force on i is
 * -dH_B/dq_i = G m_i m_j (q_j-q_i)/r^3 * (K - r K').  The direct (BS) part
 * H_A carries the pair term with 1-K (Eq. 1), weight 1-(K - r K'). */
double ora_kick_weight(double r, double rc)
{
    double K, dK;
    ora_changeover(r, rc, &K, &dK);
    return K - r * dK;
}

/* ------------------------------------------------------------------------- */
/* Critical radius, Eq. 6: rc_i = max(n1 R_H,i, n2 tau v_i).
 * [R-5] v_i = |V_i| (the body's own democratic velocity, L96);
 * R_H,i = a_i (m_i/(3 m0))^(1/3), a_i = 1/(2/r_i - V_i^2/(G m0)), and r_i in
 * place of a_i when a_i <= 0; test particles have R_H = 0.  tau enters by its
 * absolute value [R-13]. */
void ora_rcrit(int n, double G, double m0, double n1, double n2, double tau,
               const double *m, const double *q, const double *V, double *rc)
{
    for (int i = 0; i < n; ++i) {
        double x = q[i], y = q[n + i], z = q[2 * n + i];
        double vx = V[i], vy = V[n + i], vz = V[2 * n + i];
        double r = sqrt(x * x + y * y + z * z);
        double v2 = vx * vx + vy * vy + vz * vz;
        double ainv = 2.0 / r - v2 / (G * m0);
        double a = (ainv > 0.0) ? 1.0 / ainv : r;
        double rh = (m[i] > 0.0) ? a * cbrt(m[i] / (3.0 * m0)) : 0.0;
        double rv = n2 * fabs(tau) * sqrt(v2);
        double r1 = n1 * rh;
        rc[i] = (r1 > rv) ? r1 : rv;
    }
}

/* ------------------------------------------------------------------------- */
/* Kick accelerations, operator B (Eq. 2, Eq. 7 "calculate the
 * accelerations between all the bodies"), with the prechecker of L142:
 * a pair is a candidate when its separation at the kick is below 3 rc_ij,
 * rc_ij = max(rc_i, rc_j) (L92).
 * Sources j run over massive bodies only; test particles feel them but act on
 * nobody (L336-338).  Pairs are recorded as (lo,hi) index with lo massive.
 * Returns ORA_ECAPACITY if more than cap pairs would be recorded. */
int ora_accel(int n, int n_massive, double G, const double *m, const double *q,
              const double *rc, double *a, int record, int32_t *cand,
              int64_t cap, int64_t *ncand)
{
    int64_t nc = 0;
    int rcode = ORA_OK;
    for (int i = 0; i < n; ++i) {
        nsum sx = {0, 0}, sy = {0, 0}, sz = {0, 0};
        for (int j = 0; j < n_massive; ++j) {
            if (j == i) continue;
            double dx = q[j] - q[i], dy = q[n + j] - q[n + i], dz = q[2 * n + j] - q[2 * n + i];
            double r2 = dx * dx + dy * dy + dz * dz;
            double r = sqrt(r2);
            double rcij = rc[i] > rc[j] ? rc[i] : rc[j];
            double W = ora_kick_weight(r, rcij);
            double s = G * m[j] / (r2 * r) * W;
            ns_add(&sx, s * dx); ns_add(&sy, s * dy); ns_add(&sz, s * dz);
            /* each unordered pair once: (i<j both massive) or (massive j, particle i) */
            if (record && (j > i || i >= n_massive)) {
                if (r2 < 9.0 * rcij * rcij) {
                    if (nc < cap) {
                        int lo = i < j ? i : j, hi = i < j ? j : i;
                        cand[2 * nc] = lo; cand[2 * nc + 1] = hi;
                    } else rcode = ORA_ECAPACITY;
                    nc++;
                }
            }
        }
        a[i] = ns_val(&sx); a[n + i] = ns_val(&sy); a[2 * n + i] = ns_val(&sz);
    }
    if (ncand) *ncand = nc;
    return rcode;
}

/* Sun kick, operator C (Eq. 3; L108; L338 for test particles):
 * H_C = (sum p_i)^2 / 2 m0  =>  dq_i/dt = (sum_j m_j V_j)/m0 for every body,
 * the sum running over massive bodies only. */
void ora_sun_kick(int n, int n_massive, double m0, const double *m, const double *V,
                  double *q, double h)
{
    for (int c = 0; c < 3; ++c) {
        nsum s = {0, 0};
        for (int j = 0; j < n_massive; ++j) ns_add(&s, m[j] * V[c * n + j]);
        double d = h * ns_val(&s) / m0;
        for (int i = 0; i < n; ++i) q[c * n + i] += d;
    }
}

/* ------------------------------------------------------------------------- */
/* Stumpff functions c_k(x) = sum_j (-x)^j/(k+2j)!  (Danby 1988, named at L110
 * and L230).  Series for |x| <= 1, closed forms beyond. */
void ora_stumpff(double x, double c[4])
{
    if (fabs(x) <= 1.0) {
        double c2 = 0.0, c3 = 0.0, t2 = 0.5, t3 = 1.0 / 6.0;
        for (int j = 0; j < 30; ++j) {
            c2 += t2; c3 += t3;
            t2 *= -x / ((2.0 * j + 3.0) * (2.0 * j + 4.0));
            t3 *= -x / ((2.0 * j + 4.0) * (2.0 * j + 5.0));
            if (fabs(t2) < 1e-19 && fabs(t3) < 1e-19) break;
        }
        c[2] = c2; c[3] = c3; c[1] = 1.0 - x * c3; c[0] = 1.0 - x * c2;
    } else if (x > 0.0) {
        double sq = sqrt(x);
        c[0] = cos(sq); c[1] = sin(sq) / sq; c[2] = (1.0 - c[0]) / x; c[3] = (1.0 - c[1]) / x;
    } else {
        double sq = sqrt(-x);
        c[0] = cosh(sq); c[1] = sinh(sq) / sq; c[2] = (1.0 - c[0]) / x; c[3] = (1.0 - c[1]) / x;
    }
}

/* Kepler drift of one body about mu = G m0 (L114: NOT G(m0+m_i)) for time h,
 * Gauss f and g functions, Eq. 9 (L110-112), in universal variables [R-8]
 * (L230: "methods using universal variables ... (Danby 1988)").
 *   r0=|q|, u=q.V, alpha=2mu/r0-V^2;  solve  r0 s c1 + u s^2 c2 + mu s^3 c3 = h
 *   (c_k at x = alpha s^2) by Newton, dt/ds = r = r0 c0 + u s c1 + mu s^2 c2 > 0,
 *   safeguarded by bisection on the bracket the iterates establish;
 *   f = 1 - mu s^2 c2/r0, g = h - mu s^3 c3, fdot = -mu s c1/(r r0), gdot = 1 - mu s^2 c2/r.
 * Returns the iteration count (>0) or ORA_EKEPLER. */
int ora_kepler_drift(double mu, double h, double q[3], double V[3])
{
    double r0 = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2]);
    double v2 = V[0] * V[0] + V[1] * V[1] + V[2] * V[2];
    double u = q[0] * V[0] + q[1] * V[1] + q[2] * V[2];
    double alpha = 2.0 * mu / r0 - v2;
    if (h == 0.0) return 1;
    double s = h / r0, lo = -INFINITY, hi = INFINITY, c[4], r = r0;
    int it, ok = 0;
    for (it = 1; it <= 60; ++it) {
        ora_stumpff(alpha * s * s, c);
        double F = r0 * s * c[1] + u * s * s * c[2] + mu * s * s * s * c[3] - h;
        r = r0 * c[0] + u * s * c[1] + mu * s * s * c[2];
        if (F > 0.0) { if (s < hi) hi = s; } else if (F < 0.0) { if (s > lo) lo = s; }
        double ds = -F / r, sn = s + ds;
        if (!(sn > lo && sn < hi)) {
            if (isfinite(lo) && isfinite(hi)) sn = 0.5 * (lo + hi);
            else if (!isfinite(sn)) return ORA_EKEPLER;
        }
        double step = fabs(sn - s);
        s = sn;
        if (step <= 1e-15 * fabs(s)) { ok = 1; break; }
    }
    if (!ok) return ORA_EKEPLER;
    ora_stumpff(alpha * s * s, c);
    r = r0 * c[0] + u * s * c[1] + mu * s * s * c[2];
    double f = 1.0 - mu * s * s * c[2] / r0;
    double g = h - mu * s * s * s * c[3];
    double fd = -mu * s * c[1] / (r * r0);
    double gd = 1.0 - mu * s * s * c[2] / r;
    for (int k = 0; k < 3; ++k) {
        double qn = f * q[k] + g * V[k];
        double vn = fd * q[k] + gd * V[k];
        q[k] = qn; V[k] = vn;
    }
    return it;
}

int ora_drift_all(int n, double mu, double h, double *q, double *V, int64_t *iters)
{
    for (int i = 0; i < n; ++i) {
        double qq[3] = {q[i], q[n + i], q[2 * n + i]}, vv[3] = {V[i], V[n + i], V[2 * n + i]};
        int it = ora_kepler_drift(mu, h, qq, vv);
        if (it < 0) return it;
        if (iters) *iters += it;
        for (int k = 0; k < 3; ++k) { q[k * n + i] = qq[k]; V[k * n + i] = vv[k]; }
    }
    return ORA_OK;
}

/* ------------------------------------------------------------------------- */
/* Encounter search for one pair, Eq. 10-12.
 * [R-3] P = |dq|^2, Pdot = dP/dt = 2 dq.dV at the two ends of the drift.
 * [R-2] dP/dt(t) = a t^2 + b t + c with a = 6(P0-P1) + 3 h (Pd0 + Pd1) (the
 * printed minus sign at L128 contradicts Eq. 10; b and c as printed).
 * Returns Delta = min over t in [0,1] of the Hermite cubic: the smaller end
 * value and the cubic at every real critical point inside (0,1). */
static double hermite_P(double t, double P0, double P1, double Pd0, double Pd1, double h)
{   /* Eq. 12 (L139) */
    return (1 - t) * (1 - t) * (1 + 2 * t) * P0 + t * t * (3 - 2 * t) * P1
         + t * (1 - t) * (1 - t) * h * Pd0 - t * t * (1 - t) * h * Pd1;
}
double ora_hermite_min(double P0, double P1, double Pd0, double Pd1, double h)
{
    double a = 6.0 * (P0 - P1) + 3.0 * h * (Pd0 + Pd1);
    double b = 6.0 * (P1 - P0) - 2.0 * h * (2.0 * Pd0 + Pd1);
    double c = h * Pd0;
    double D = P0 < P1 ? P0 : P1;
    double t[2]; int nt = 0;
    if (a == 0.0) { if (b != 0.0) t[nt++] = -c / b; }
    else {
        double disc = b * b - 4.0 * a * c;
        if (disc >= 0.0) {
            double sq = sqrt(disc);
            double qq = -0.5 * (b + (b >= 0.0 ? sq : -sq));
            t[nt++] = qq / a;
            if (qq != 0.0) t[nt++] = c / qq;
        }
    }
    for (int k = 0; k < nt; ++k)
        if (t[k] > 0.0 && t[k] < 1.0) {
            double P = hermite_P(t[k], P0, P1, Pd0, Pd1, h);
            if (P < D) D = P;
        }
    return D;
}

/* Confirm candidates (L159, L200, L276-278): encounter iff Delta < rc_ij^2.
 * q0,V0 = state before the drift, q1,V1 = after (L122). */
int ora_confirm(int n, const double *q0, const double *V0, const double *q1, const double *V1,
                const double *rc, double h, const int32_t *cand, int64_t ncand,
                int32_t *enc, int64_t cap, int64_t *nenc)
{
    int64_t ne = 0; int rcode = ORA_OK;
    for (int64_t e = 0; e < ncand; ++e) {
        int i = cand[2 * e], j = cand[2 * e + 1];
        double P[2], Pd[2];
        const double *qs[2] = {q0, q1}, *vs[2] = {V0, V1};
        for (int k = 0; k < 2; ++k) {
            double dx = qs[k][j] - qs[k][i], dy = qs[k][n + j] - qs[k][n + i], dz = qs[k][2 * n + j] - qs[k][2 * n + i];
            double dvx = vs[k][j] - vs[k][i], dvy = vs[k][n + j] - vs[k][n + i], dvz = vs[k][2 * n + j] - vs[k][2 * n + i];
            P[k] = dx * dx + dy * dy + dz * dz;
            Pd[k] = 2.0 * (dx * dvx + dy * dvy + dz * dvz);
        }
        double rcij = rc[i] > rc[j] ? rc[i] : rc[j];
        double D = ora_hermite_min(P[0], P[1], Pd[0], Pd[1], h);
        if (D < rcij * rcij) {
            if (ne < cap) { enc[2 * ne] = i; enc[2 * ne + 1] = j; } else rcode = ORA_ECAPACITY;
            ne++;
        }
    }
    *nenc = ne;
    return rcode;
}

/* ------------------------------------------------------------------------- */
/* Group finding, PAPER.md Appendix: LINK[i]=i; repeat
 *   LINK[P1[e]] = min(LINK[P1[e]], LINK[P2[e]]); LINK[P2[e]] = min(same);
 *   LINK[i] = LINK[LINK[i]]
 * until LINK is unchanged.  LINK[i] is then the lowest index in i's group. */
void ora_group(int n, const int32_t *pairs, int64_t npairs, int32_t *link)
{
    for (int i = 0; i < n; ++i) link[i] = i;
    int changed = 1;
    while (changed) {
        changed = 0;
        for (int64_t e = 0; e < npairs; ++e) {
            int p1 = pairs[2 * e], p2 = pairs[2 * e + 1];
            int mn = link[p1] < link[p2] ? link[p1] : link[p2];
            if (link[p1] != mn) { link[p1] = mn; changed = 1; }
            if (link[p2] != mn) { link[p2] = mn; changed = 1; }
        }
        for (int i = 0; i < n; ++i)
            if (link[i] != link[link[i]]) { link[i] = link[link[i]]; changed = 1; }
    }
}

/* ------------------------------------------------------------------------- */
/* Direct integration of H_A for one encounter group (Eq. 1; L116; L314:
 * the star is fixed at the origin during the step; L505: every pair inside the
 * group interacts, indirect ones included).
 * Right-hand side: qdot = V, Vdot = -G m0 q/|q|^3
 *                  + sum_{j in group, massive} G m_j (q_j-q_i)/r^3 (1 - W(r, rc_ij)). */
static void bs_rhs(int ng, double G, double m0, const double *m, const double *rc,
                   const double *q, double *acc)
{
    for (int i = 0; i < ng; ++i) {
        double x = q[i], y = q[ng + i], z = q[2 * ng + i];
        double r2 = x * x + y * y + z * z, r = sqrt(r2);
        double s0 = -G * m0 / (r2 * r);
        nsum sx = {0, 0}, sy = {0, 0}, sz = {0, 0};
        ns_add(&sx, s0 * x); ns_add(&sy, s0 * y); ns_add(&sz, s0 * z);
        for (int j = 0; j < ng; ++j) {
            if (j == i || m[j] == 0.0) continue;
            double dx = q[j] - x, dy = q[ng + j] - y, dz = q[2 * ng + j] - z;
            double d2 = dx * dx + dy * dy + dz * dz, d = sqrt(d2);
            double rcij = rc[i] > rc[j] ? rc[i] : rc[j];
            double w = 1.0 - ora_kick_weight(d, rcij);
            if (w == 0.0) continue;
            double s = G * m[j] / (d2 * d) * w;
            ns_add(&sx, s * dx); ns_add(&sy, s * dy); ns_add(&sz, s * dz);
        }
        acc[i] = ns_val(&sx); acc[ng + i] = ns_val(&sy); acc[2 * ng + i] = ns_val(&sz);
    }
}

/* Gragg's modified midpoint rule over H with nsub substeps (Hairer et al.,
 * cited L116/L615): z1 = z0 + eta f(z0); z_{m+1} = z_{m-1} + 2 eta f(z_m);
 * result = (z_n + z_{n-1} + eta f(z_n))/2.  acc0 = f(z0) is shared. */
static void bs_midpoint(int ng, double G, double m0, const double *m, const double *rc,
                        const double *q0, const double *V0, const double *acc0,
                        double H, int nsub, double *qo, double *Vo, double *work)
{
    int N3 = 3 * ng;
    double eta = H / nsub;
    double *qa = work, *Va = work + N3, *qb = work + 2 * N3, *Vb = work + 3 * N3, *acc = work + 4 * N3;
    for (int k = 0; k < N3; ++k) {
        qa[k] = q0[k]; Va[k] = V0[k];
        qb[k] = q0[k] + eta * V0[k]; Vb[k] = V0[k] + eta * acc0[k];
    }
    for (int mstep = 1; mstep < nsub; ++mstep) {
        bs_rhs(ng, G, m0, m, rc, qb, acc);
        for (int k = 0; k < N3; ++k) {
            double qn = qa[k] + 2.0 * eta * Vb[k];
            double vn = Va[k] + 2.0 * eta * acc[k];
            qa[k] = qb[k]; Va[k] = Vb[k]; qb[k] = qn; Vb[k] = vn;
        }
    }
    bs_rhs(ng, G, m0, m, rc, qb, acc);
    for (int k = 0; k < N3; ++k) {
        qo[k] = 0.5 * (qb[k] + qa[k] + eta * Vb[k]);
        Vo[k] = 0.5 * (Vb[k] + Va[k] + eta * acc[k]);
    }
}

/* Bulirsch-Stoer over the whole drift interval h for one group [R-7]:
 * substep sequence n_k = 2,4,...,16; Aitken-Neville extrapolation in (H/n_k)^2,
 * T[k][j] = T[k][j-1] + (T[k][j-1]-T[k-1][j-1])/((n_k/n_{k-j})^2 - 1);
 * error^2 = max over bodies of max(|dq_i|^2/|q_i|^2, |dV_i|^2/|V_i|^2),
 * d = T[k][k]-T[k][k-1], scales taken at the start of the BS step; accept when
 * error <= eps.  First trial H = h; after 8 columns without convergence H <- H/2;
 * after an accept with k <= 4 (at most five columns) H <- 1.5 H; H is cut to
 * land exactly on h; ORA_EBS when |H| < 1e-12 |h|.
 * q,V: [3*ng] SoA, overwritten.  stats[0] += BS steps, stats[1] += RHS calls. */
#define BS_KMAX 8

/* Collisions (L316-328, section 3.2.7).  "To find collisions between the Bulirsch-Stoer time steps, we use the same
 * code as in the close encounter detection" (L328): after every ACCEPTED Bulirsch-Stoer step of a group the minimum of
 * the cubic Hermite interpolant of the squared separation (Eq. 10-12) over that step is compared, pair by pair, with
 * (R_i + R_j)^2.  A colliding pair merges as perfectly inelastic bodies at the END of that step [reading R-19]:
 *   m = m_i + m_j, q = (m_i q_i + m_j q_j)/m, V = (m_i V_i + m_j V_j)/m   (linear momentum conserved, L316),
 *   R = (R_i^3 + R_j^3)^(1/3)                                             [R-20: the paper does not say; same density],
 *   U += 1/2 m_i m_j/(m_i + m_j) v_ij^2 - G m_i m_j / r_ij                (L318-322, at the merge state),
 *   spin += spin_i + spin_j + m_i m_j/m (q_i - q_j) x (V_i - V_j)          (angular momentum conservation, L324),
 * the new body keeps the index of the more massive one, the smaller index if the masses are equal (L324); the other
 * becomes a massless ghost (L324) and is parked on a circular orbit of radius 1000 (index + 1) about the star, where
 * it meets nothing and adds exact zeros to every sum [R-21: "removed later" -- the caller compacts].  A test particle
 * that hits a massive body is reported and removed, with no effect on the body (L336); particles do not collide with
 * each other.  Pairs are visited in the order of the group's member list (a < b); a body removed earlier in the
 * same step is skipped.  The report holds the two states at the START of that Bulirsch-Stoer step, "the last time
 * step before the collision happens" (L326).  The integration of the group then goes on from the merged state. */
#define ORA_EV 24                 /* doubles per event record */
typedef struct {
    int enabled;
    const int *gidx;              /* global index of every member */
    const int *kind;              /* 0 massive, 1 test particle, 2 removed (updated here) */
    double *R;                    /* physical radii of the members (updated) */
    double *mm;                   /* masses of the members (updated; the const m passed to the integrator is this array) */
    double *spin;                 /* [3 ng] spins of the members (updated) */
    double *U;                    /* internal energy accumulator */
    double *ev; int64_t *nev, evcap;   /* event records */
    double step_id;
    int *kindw;                   /* writable alias of kind */
} ora_coll;

double ora_hermite_min(double P0, double P1, double Pd0, double Pd1, double h);

static void coll_scan(int ng, double G, double m0, ora_coll *cc, const double *q0, const double *V0,
                      double *q1, double *V1, double H)
{
    for (int a = 0; a < ng; ++a)
        for (int b = a + 1; b < ng; ++b) {
            if (cc->kindw[a] == 2 || cc->kindw[b] == 2) continue;
            if (cc->kindw[a] == 1 && cc->kindw[b] == 1) continue;            /* particles do not see each other (L336) */
            double d0[3], w0[3], d1[3], w1[3];
            for (int c = 0; c < 3; ++c) {
                d0[c] = q0[c * ng + b] - q0[c * ng + a]; w0[c] = V0[c * ng + b] - V0[c * ng + a];
                d1[c] = q1[c * ng + b] - q1[c * ng + a]; w1[c] = V1[c * ng + b] - V1[c * ng + a];
            }
            double P0 = d0[0] * d0[0] + d0[1] * d0[1] + d0[2] * d0[2], Pd0 = 2.0 * (d0[0] * w0[0] + d0[1] * w0[1] + d0[2] * w0[2]);
            double P1 = d1[0] * d1[0] + d1[1] * d1[1] + d1[2] * d1[2], Pd1 = 2.0 * (d1[0] * w1[0] + d1[1] * w1[1] + d1[2] * w1[2]);
            double D = ora_hermite_min(P0, P1, Pd0, Pd1, H);
            double Rs = cc->R[a] + cc->R[b];
            if (!(D < Rs * Rs)) continue;
            /* survivor s, removed d */
            int sv = a, dd = b, kindev = 0;
            if (cc->kindw[a] == 1) { sv = b; dd = a; kindev = 1; }
            else if (cc->kindw[b] == 1) { sv = a; dd = b; kindev = 1; }
            else if (cc->mm[b] > cc->mm[a]) { sv = b; dd = a; }               /* equal masses: the smaller index (a) */
            double ma = cc->mm[sv], mb = cc->mm[dd], mt = ma + mb, Uev = 0.0;
            if (*cc->nev < cc->evcap) {
                double *e = cc->ev + ORA_EV * (*cc->nev);
                e[0] = cc->step_id; e[1] = kindev; e[2] = cc->gidx[sv]; e[3] = cc->gidx[dd];
                e[4] = ma; e[5] = mb; e[6] = cc->R[sv]; e[7] = cc->R[dd];
                for (int c = 0; c < 3; ++c) {
                    e[8 + c] = q0[c * ng + sv]; e[11 + c] = V0[c * ng + sv];
                    e[14 + c] = q0[c * ng + dd]; e[17 + c] = V0[c * ng + dd];
                }
            }
            if (kindev == 0) {
                double dq[3], dv[3], r2 = 0.0, v2 = 0.0;
                for (int c = 0; c < 3; ++c) {
                    dq[c] = q1[c * ng + sv] - q1[c * ng + dd]; dv[c] = V1[c * ng + sv] - V1[c * ng + dd];
                    r2 += dq[c] * dq[c]; v2 += dv[c] * dv[c];
                }
                double mu = ma * mb / mt;
                Uev = 0.5 * mu * v2 - G * ma * mb / sqrt(r2);
                *cc->U += Uev;
                double lx = mu * (dq[1] * dv[2] - dq[2] * dv[1]), ly = mu * (dq[2] * dv[0] - dq[0] * dv[2]), lz = mu * (dq[0] * dv[1] - dq[1] * dv[0]);
                cc->spin[sv] += cc->spin[dd] + lx; cc->spin[ng + sv] += cc->spin[ng + dd] + ly; cc->spin[2 * ng + sv] += cc->spin[2 * ng + dd] + lz;
                for (int c = 0; c < 3; ++c) {
                    q1[c * ng + sv] = (ma * q1[c * ng + sv] + mb * q1[c * ng + dd]) / mt;
                    V1[c * ng + sv] = (ma * V1[c * ng + sv] + mb * V1[c * ng + dd]) / mt;
                }
                cc->R[sv] = cbrt(cc->R[sv] * cc->R[sv] * cc->R[sv] + cc->R[dd] * cc->R[dd] * cc->R[dd]);
                cc->mm[sv] = mt;
            }
            if (*cc->nev < cc->evcap) {
                double *e = cc->ev + ORA_EV * (*cc->nev);
                e[20] = Uev; e[21] = cc->spin[sv]; e[22] = cc->spin[ng + sv]; e[23] = cc->spin[2 * ng + sv];
            }
            ++*cc->nev;
            /* the ghost: massless, parked far away on a circular orbit */
            double Rp = 1000.0 * (double)(cc->gidx[dd] + 1);
            cc->mm[dd] = 0.0; cc->R[dd] = 0.0; cc->kindw[dd] = 2;
            cc->spin[dd] = cc->spin[ng + dd] = cc->spin[2 * ng + dd] = 0.0;
            q1[dd] = Rp; q1[ng + dd] = 0.0; q1[2 * ng + dd] = 0.0;
            V1[dd] = 0.0; V1[ng + dd] = sqrt(G * m0 / Rp); V1[2 * ng + dd] = 0.0;
        }
}

static int bs_group_impl(int ng, double G, double m0, const double *m, const double *rc,
                         double *q, double *V, double h, double eps, int64_t *stats, ora_coll *cc);

int ora_bs_group(int ng, double G, double m0, const double *m, const double *rc,
                 double *q, double *V, double h, double eps, int64_t *stats)
{
    return bs_group_impl(ng, G, m0, m, rc, q, V, h, eps, stats, NULL);
}

static int bs_group_impl(int ng, double G, double m0, const double *m, const double *rc,
                         double *q, double *V, double h, double eps, int64_t *stats, ora_coll *cc)
{
    int N3 = 3 * ng, N6 = 6 * ng;
    if (h == 0.0 || ng == 0) return ORA_OK;
    double *T = (double *)malloc(sizeof(double) * (size_t)(BS_KMAX * BS_KMAX) * N6);
    double *work = (double *)malloc(sizeof(double) * 5 * N3);
    double *acc0 = (double *)malloc(sizeof(double) * N3);
    double *sq = (double *)malloc(sizeof(double) * 2 * ng);
    int rcode = ORA_OK;
    double done = 0.0, H = h;
    int last = 0;
    while (!last) {
        double rem = h - done;
        if (fabs(H) >= fabs(rem)) { H = rem; last = 1; }
        for (int i = 0; i < ng; ++i) {
            sq[i] = q[i] * q[i] + q[ng + i] * q[ng + i] + q[2 * ng + i] * q[2 * ng + i];
            sq[ng + i] = V[i] * V[i] + V[ng + i] * V[ng + i] + V[2 * ng + i] * V[2 * ng + i];
        }
        bs_rhs(ng, G, m0, m, rc, q, acc0);
        if (stats) stats[1] += 1;
        int accepted = 0;
        while (!accepted) {
            for (int k = 0; k < BS_KMAX && !accepted; ++k) {
                int nk = 2 * (k + 1);
                double *Tk0 = T + (size_t)(k * BS_KMAX) * N6;
                bs_midpoint(ng, G, m0, m, rc, q, V, acc0, H, nk, Tk0, Tk0 + N3, work);
                if (stats) stats[1] += nk;
                for (int j = 1; j <= k; ++j) {
                    double ratio = (double)nk / (double)(2 * (k - j + 1));
                    double den = ratio * ratio - 1.0;
                    double *Tkj = T + (size_t)(k * BS_KMAX + j) * N6;
                    double *Tkj1 = T + (size_t)(k * BS_KMAX + j - 1) * N6;
                    double *Tk1j1 = T + (size_t)((k - 1) * BS_KMAX + j - 1) * N6;
                    for (int e = 0; e < N6; ++e) Tkj[e] = Tkj1[e] + (Tkj1[e] - Tk1j1[e]) / den;
                }
                if (k >= 1) {
                    double *Tkk = T + (size_t)(k * BS_KMAX + k) * N6;
                    double *Tkk1 = T + (size_t)(k * BS_KMAX + k - 1) * N6;
                    double err2 = 0.0;
                    for (int i = 0; i < ng; ++i) {
                        double dq2 = 0.0, dv2 = 0.0;
                        for (int c = 0; c < 3; ++c) {
                            double dq = Tkk[c * ng + i] - Tkk1[c * ng + i];
                            double dv = Tkk[N3 + c * ng + i] - Tkk1[N3 + c * ng + i];
                            dq2 += dq * dq; dv2 += dv * dv;
                        }
                        double e1 = dq2 / sq[i], e2 = dv2 / sq[ng + i];
                        if (e1 > err2) err2 = e1;
                        if (e2 > err2) err2 = e2;
                    }
                    if (err2 <= eps * eps) {
                        if (cc && cc->enabled) coll_scan(ng, G, m0, cc, q, V, Tkk, Tkk + N3, H);   /* may merge bodies in Tkk */
                        memcpy(q, Tkk, sizeof(double) * N3);
                        memcpy(V, Tkk + N3, sizeof(double) * N3);
                        done += H;
                        if (stats) stats[0] += 1;
                        if (k <= 4) H *= 1.5;
                        accepted = 1;
                    }
                }
            }
            if (!accepted) {
                H *= 0.5; last = 0;
                if (fabs(H) < 1e-12 * fabs(h)) { rcode = ORA_EBS; goto out; }
            }
        }
    }
out:
    free(T); free(work); free(acc0); free(sq);
    return rcode;
}

/* One group with collisions, for the pins: kind[ng] (0 massive, 1 test particle, 2 removed), R[ng], spin[3 ng], m[ng]
 * are updated; events are appended to ev (ORA_EV doubles each, member numbers as indices). */
int ora_bs_group_collide(int ng, double G, double m0, double *m, const double *rc, double *R, int32_t *kind, double *spin,
                         double *q, double *V, double h, double eps, double *U, double *ev, int64_t evcap, int64_t *nev)
{
    int *gidx = (int *)malloc(sizeof(int) * (size_t)ng), *k2 = (int *)malloc(sizeof(int) * (size_t)ng);
    for (int i = 0; i < ng; ++i) { gidx[i] = i; k2[i] = kind[i]; }
    ora_coll cc;
    memset(&cc, 0, sizeof cc);
    cc.enabled = 1; cc.gidx = gidx; cc.kind = k2; cc.kindw = k2; cc.R = R; cc.mm = m; cc.spin = spin;
    cc.U = U; cc.ev = ev; cc.nev = nev; cc.evcap = evcap; cc.step_id = 0.0;
    int rcode = bs_group_impl(ng, G, m0, m, rc, q, V, h, eps, NULL, &cc);
    for (int i = 0; i < ng; ++i) kind[i] = k2[i];
    free(gidx); free(k2);
    return rcode;
}

/* ------------------------------------------------------------------------- */
/* Energy and angular momentum in democratic coordinates: H = H_A+H_B+H_C of
 * Eq. 1-3 (L73-80) with the K terms cancelling:
 *   E = sum m V^2/2 + (sum m V)^2/(2 m0) - sum G m0 m/r - sum_{i<j} G m_i m_j/r_ij
 *   L = sum m q x V.
 * parts[0..2] = H_A, H_B, H_C evaluated separately with the changeover (needs rc). */
void ora_energy(int n_massive, int n, double G, double m0, const double *m,
                const double *q, const double *V, const double *rc,
                double *E, double *L, double *parts)
{
    nsum kin = {0, 0}, pot0 = {0, 0}, potp = {0, 0}, hbK = {0, 0};
    nsum px = {0, 0}, py = {0, 0}, pz = {0, 0}, lx = {0, 0}, ly = {0, 0}, lz = {0, 0};
    for (int i = 0; i < n_massive; ++i) {
        double x = q[i], y = q[n + i], z = q[2 * n + i], vx = V[i], vy = V[n + i], vz = V[2 * n + i];
        ns_add(&kin, 0.5 * m[i] * (vx * vx + vy * vy + vz * vz));
        ns_add(&pot0, -G * m0 * m[i] / sqrt(x * x + y * y + z * z));
        ns_add(&px, m[i] * vx); ns_add(&py, m[i] * vy); ns_add(&pz, m[i] * vz);
        ns_add(&lx, m[i] * (y * vz - z * vy)); ns_add(&ly, m[i] * (z * vx - x * vz)); ns_add(&lz, m[i] * (x * vy - y * vx));
        for (int j = i + 1; j < n_massive; ++j) {
            double dx = q[j] - x, dy = q[n + j] - y, dz = q[2 * n + j] - z;
            double r = sqrt(dx * dx + dy * dy + dz * dz);
            double t = -G * m[i] * m[j] / r;
            ns_add(&potp, t);
            if (rc) {
                double K, dK, rcij = rc[i] > rc[j] ? rc[i] : rc[j];
                ora_changeover(r, rcij, &K, &dK);
                ns_add(&hbK, t * K);
            }
        }
    }
    double P2 = ns_val(&px) * ns_val(&px) + ns_val(&py) * ns_val(&py) + ns_val(&pz) * ns_val(&pz);
    double HC = P2 / (2.0 * m0);
    *E = ns_val(&kin) + HC + ns_val(&pot0) + ns_val(&potp);
    if (L) { L[0] = ns_val(&lx); L[1] = ns_val(&ly); L[2] = ns_val(&lz); }
    if (parts) {
        double HB = rc ? ns_val(&hbK) : ns_val(&potp);
        parts[1] = HB; parts[2] = HC;
        parts[0] = ns_val(&kin) + ns_val(&pot0) + (ns_val(&potp) - HB);
    }
}

/* Heliocentric (x, v) <-> democratic (q = x, V = barycentric v), L69.
 * V_i = v_i - sum m_j v_j/(m0 + sum m_j);  v_i = V_i + sum m_j V_j/m0. */
void ora_helio_to_demo(int n, int n_massive, double m0, const double *m, const double *v, double *V)
{
    double mt = m0;
    for (int j = 0; j < n_massive; ++j) mt += m[j];
    for (int c = 0; c < 3; ++c) {
        nsum s = {0, 0};
        for (int j = 0; j < n_massive; ++j) ns_add(&s, m[j] * v[c * n + j]);
        double d = ns_val(&s) / mt;
        for (int i = 0; i < n; ++i) V[c * n + i] = v[c * n + i] - d;
    }
}
void ora_demo_to_helio(int n, int n_massive, double m0, const double *m, const double *V, double *v)
{
    for (int c = 0; c < 3; ++c) {
        nsum s = {0, 0};
        for (int j = 0; j < n_massive; ++j) ns_add(&s, m[j] * V[c * n + j]);
        double d = ns_val(&s) / m0;
        for (int i = 0; i < n; ++i) v[c * n + i] = V[c * n + i] + d;
    }
}

/* ------------------------------------------------------------------------- */
/* One system (one star).  Multi-simulation mode (L344-376) is a loop over
 * independent ora_sys objects. */
typedef struct {
    int n, n_massive;
    double G, m0, n1, n2, bs_eps;
    int cull;                 /* 1: prechecker (L142); 0: every pair goes through Eq. 12 [R-9] */
    double *m, *q, *V, *rc;   /* [n], [3n], [3n], [n] */
    double *q0, *V0, *a;      /* pre-drift copy, accelerations */
    int64_t cap, n_cand, n_enc;
    int32_t *cand, *enc, *label;
    int64_t stat_kepler_iters, stat_bs[2], stat_force_evals, stat_groups, stat_maxgroup;
    /* collisions, ejections, removal (L316-332, L336, L378-384); off unless ora_set_collisions() switches them on */
    int coll;                 /* 1: collisions are looked for between the Bulirsch-Stoer steps */
    double rcut, rcut_sun;    /* ejection limits (L330-332); 0 = none */
    int nmin;                 /* the system is stopped when fewer bodies are left (L378-384); 0 = never */
    double *R, *spin;         /* [n] physical radii, [3n] spins */
    int *kind;                /* [n] 0 massive, 1 test particle, 2 removed */
    double U;                 /* internal energy of the collisions so far (L318-322) */
    double *ev; int64_t nev, evcap;
    int64_t step_id;
} ora_sys;

ora_sys *ora_create(int n, int n_massive, double G, double m0, double n1, double n2,
                    double bs_eps, int64_t cap)
{
    if (n <= 0 || n_massive < 0 || n_massive > n) return NULL;
    ora_sys *s = (ora_sys *)calloc(1, sizeof(ora_sys));
    s->n = n; s->n_massive = n_massive; s->G = G; s->m0 = m0; s->n1 = n1; s->n2 = n2;
    s->bs_eps = bs_eps; s->cull = 1; s->cap = cap;
    s->m = (double *)calloc(n, 8); s->rc = (double *)calloc(n, 8);
    s->q = (double *)calloc(3 * (size_t)n, 8); s->V = (double *)calloc(3 * (size_t)n, 8);
    s->q0 = (double *)calloc(3 * (size_t)n, 8); s->V0 = (double *)calloc(3 * (size_t)n, 8);
    s->a = (double *)calloc(3 * (size_t)n, 8);
    s->cand = (int32_t *)calloc(2 * (size_t)cap, 4); s->enc = (int32_t *)calloc(2 * (size_t)cap, 4);
    s->label = (int32_t *)calloc(n, 4);
    s->R = (double *)calloc(n, 8); s->spin = (double *)calloc(3 * (size_t)n, 8);
    s->kind = (int *)calloc(n, sizeof(int));
    for (int i = n_massive; i < n; ++i) s->kind[i] = 1;
    s->evcap = 4096; s->ev = (double *)calloc((size_t)s->evcap * ORA_EV, 8);
    return s;
}
void ora_destroy(ora_sys *s)
{
    if (!s) return;
    free(s->m); free(s->rc); free(s->q); free(s->V); free(s->q0); free(s->V0); free(s->a);
    free(s->cand); free(s->enc); free(s->label); free(s->R); free(s->spin); free(s->kind); free(s->ev); free(s);
}
/* radii [n]; coll: look for collisions; rcut, rcut_sun: ejection limits (0 = none); nmin: stop limit (0 = never) */
void ora_set_collisions(ora_sys *s, const double *R, int coll, double rcut, double rcut_sun, int nmin)
{
    if (R) memcpy(s->R, R, 8 * (size_t)s->n);
    s->coll = coll; s->rcut = rcut; s->rcut_sun = rcut_sun; s->nmin = nmin;
}
int64_t ora_get_events(const ora_sys *s, double *buf, int64_t cap)
{
    int64_t k = s->nev < s->evcap ? s->nev : s->evcap;
    if (k > cap) k = cap;
    if (buf && k > 0) memcpy(buf, s->ev, 8 * (size_t)k * ORA_EV);
    return s->nev;
}
void ora_get_bodies(const ora_sys *s, double *m, double *R, int32_t *kind, double *spin)
{
    if (m) memcpy(m, s->m, 8 * (size_t)s->n);
    if (R) memcpy(R, s->R, 8 * (size_t)s->n);
    if (kind) for (int i = 0; i < s->n; ++i) kind[i] = s->kind[i];
    if (spin) memcpy(spin, s->spin, 24 * (size_t)s->n);
}
double ora_internal_energy(const ora_sys *s) { return s->U; }
void ora_set_cull(ora_sys *s, int cull) { s->cull = cull; }

/* x, v heliocentric, SoA [3n] */
void ora_set_state(ora_sys *s, const double *m, const double *x, const double *v)
{
    memcpy(s->m, m, 8 * (size_t)s->n);
    memcpy(s->q, x, 24 * (size_t)s->n);
    ora_helio_to_demo(s->n, s->n_massive, s->m0, s->m, v, s->V);
}
void ora_get_state(const ora_sys *s, double *x, double *v)
{
    memcpy(x, s->q, 24 * (size_t)s->n);
    ora_demo_to_helio(s->n, s->n_massive, s->m0, s->m, s->V, v);
}
void ora_get_demo(const ora_sys *s, double *q, double *V, double *rc)
{
    memcpy(q, s->q, 24 * (size_t)s->n); memcpy(V, s->V, 24 * (size_t)s->n);
    if (rc) memcpy(rc, s->rc, 8 * (size_t)s->n);
}
void ora_set_demo(ora_sys *s, const double *q, const double *V)
{
    memcpy(s->q, q, 24 * (size_t)s->n); memcpy(s->V, V, 24 * (size_t)s->n);
}

static int kick(ora_sys *s, double h, int record)
{
    int rcode = ora_accel(s->n, s->n_massive, s->G, s->m, s->q, s->rc, s->a, record,
                          s->cand, s->cap, record ? &s->n_cand : NULL);
    s->stat_force_evals++;
    for (size_t k = 0; k < 3 * (size_t)s->n; ++k) s->V[k] += h * s->a[k];
    return rcode;
}

/* All pairs with at least one massive member, for the no-cull mode [R-9]. */
static int all_pairs(ora_sys *s)
{
    int64_t nc = 0;
    for (int i = 0; i < s->n_massive; ++i)
        for (int j = i + 1; j < s->n; ++j) {
            if (nc >= s->cap) return ORA_ECAPACITY;
            s->cand[2 * nc] = i; s->cand[2 * nc + 1] = j; nc++;
        }
    s->n_cand = nc;
    return ORA_OK;
}

/* BS for the groups found in this substep (L161-163, L342).
 * Massive groups: connected components of the massive-massive encounter graph,
 * all members integrated from the pre-drift state and overwritten (L163).
 * Test particle p with encounters [R-12]: group = {p} + every massive body it
 * meets + those bodies' massive groups; integrated from the pre-drift state,
 * only p is written back (L342). */
static int do_groups(ora_sys *s, double h)
{
    int n = s->n, nm = s->n_massive, rcode = ORA_OK;
    /* massive-massive pairs first */
    int32_t *mm = (int32_t *)malloc(8 * (size_t)(s->n_enc + 1));
    int64_t nmm = 0;
    for (int64_t e = 0; e < s->n_enc; ++e)
        if (s->enc[2 * e + 1] < nm) { mm[2 * nmm] = s->enc[2 * e]; mm[2 * nmm + 1] = s->enc[2 * e + 1]; nmm++; }
    ora_group(n, mm, nmm, s->label);
    free(mm);
    int *idx = (int *)malloc(sizeof(int) * (size_t)(nm + 1));
    double *gm = (double *)malloc(8 * (size_t)(nm + 1)), *grc = (double *)malloc(8 * (size_t)(nm + 1));
    double *gq = (double *)malloc(24 * (size_t)(nm + 1)), *gV = (double *)malloc(24 * (size_t)(nm + 1));
    /* collisions: every group starts from the bodies as they were before this substep's groups were integrated (a particle's
       group re-integrates the massive bodies it contains, merges included, and must see them unmerged) */
    double *gR = (double *)malloc(8 * (size_t)(nm + 1)), *gspin = (double *)malloc(24 * (size_t)(nm + 1));
    int *gkind = (int *)malloc(sizeof(int) * (size_t)(nm + 1));
    double *m_pre = (double *)malloc(8 * (size_t)n), *R_pre = (double *)malloc(8 * (size_t)n), *spin_pre = (double *)malloc(24 * (size_t)n);
    int *kind_pre = (int *)malloc(sizeof(int) * (size_t)n);
    memcpy(m_pre, s->m, 8 * (size_t)n); memcpy(R_pre, s->R, 8 * (size_t)n); memcpy(spin_pre, s->spin, 24 * (size_t)n);
    memcpy(kind_pre, s->kind, sizeof(int) * (size_t)n);
    ora_coll cc;
    memset(&cc, 0, sizeof cc);
    cc.enabled = s->coll; cc.gidx = idx; cc.kind = gkind; cc.kindw = gkind; cc.R = gR; cc.mm = gm; cc.spin = gspin;
    cc.U = &s->U; cc.ev = s->ev; cc.nev = &s->nev; cc.evcap = s->evcap; cc.step_id = (double)s->step_id;
    /* results of massive groups are collected first and written after the
       particle groups have read the pre-drift state (they only use q0,V0). */
    for (int root = 0; root < nm && rcode == ORA_OK; ++root) {
        if (s->label[root] != root) continue;
        int ng = 0;
        for (int i = root; i < nm; ++i) if (s->label[i] == root) idx[ng++] = i;
        if (ng < 2) continue;
        for (int k = 0; k < ng; ++k) {
            gm[k] = m_pre[idx[k]]; grc[k] = s->rc[idx[k]]; gR[k] = R_pre[idx[k]]; gkind[k] = kind_pre[idx[k]];
            for (int c = 0; c < 3; ++c) {
                gq[c * ng + k] = s->q0[c * n + idx[k]]; gV[c * ng + k] = s->V0[c * n + idx[k]];
                gspin[c * ng + k] = spin_pre[c * n + idx[k]];
            }
        }
        rcode = bs_group_impl(ng, s->G, s->m0, gm, grc, gq, gV, h, s->bs_eps, s->stat_bs, &cc);
        for (int k = 0; k < ng; ++k) {
            for (int c = 0; c < 3; ++c) {
                s->q[c * n + idx[k]] = gq[c * ng + k]; s->V[c * n + idx[k]] = gV[c * ng + k];
                s->spin[c * n + idx[k]] = gspin[c * ng + k];
            }
            s->m[idx[k]] = gm[k]; s->R[idx[k]] = gR[k]; s->kind[idx[k]] = gkind[k];
        }
        s->stat_groups++;
        if (ng > s->stat_maxgroup) s->stat_maxgroup = ng;
    }
    /* test particles */
    if (n > nm && rcode == ORA_OK) {
        char *in = (char *)malloc((size_t)nm + 1);
        int64_t *head = (int64_t *)malloc(8 * (size_t)(n - nm)), *next = (int64_t *)malloc(8 * (size_t)(s->n_enc + 1));
        for (int p = nm; p < n; ++p) { head[p - nm] = -1; s->label[p] = p; }
        for (int64_t e = s->n_enc - 1; e >= 0; --e)
            if (s->enc[2 * e + 1] >= nm) { int p = s->enc[2 * e + 1]; next[e] = head[p - nm]; head[p - nm] = e; }
        for (int p = nm; p < n && rcode == ORA_OK; ++p) {
            if (head[p - nm] < 0) continue;
            int lab = p;
            memset(in, 0, (size_t)nm);
            for (int64_t e = head[p - nm]; e >= 0; e = next[e]) {
                int root = s->label[s->enc[2 * e]];
                for (int i = 0; i < nm; ++i) if (s->label[i] == root) in[i] = 1;
                if (root < lab) lab = root;
            }
            s->label[p] = lab;
            int ng = 0;
            for (int i = 0; i < nm; ++i) if (in[i]) idx[ng++] = i;
            idx[ng++] = p;
            for (int k = 0; k < ng; ++k) {
                gm[k] = m_pre[idx[k]]; grc[k] = s->rc[idx[k]]; gR[k] = R_pre[idx[k]]; gkind[k] = kind_pre[idx[k]];
                for (int c = 0; c < 3; ++c) {
                    gq[c * ng + k] = s->q0[c * n + idx[k]]; gV[c * ng + k] = s->V0[c * n + idx[k]];
                    gspin[c * ng + k] = spin_pre[c * n + idx[k]];
                }
            }
            /* the massive bodies' own collisions were reported (and their energy counted) by their massive group: here
               they are only re-enacted; the particle's collision is new */
            double U_dummy = 0.0;
            int64_t nev0 = s->nev;
            cc.U = &U_dummy;
            rcode = bs_group_impl(ng, s->G, s->m0, gm, grc, gq, gV, h, s->bs_eps, s->stat_bs, &cc);
            cc.U = &s->U;
            {   /* keep only the particle's events of this group */
                int64_t w = nev0;
                for (int64_t e = nev0; e < s->nev && e < s->evcap; ++e)
                    if (s->ev[ORA_EV * e + 1] == 1.0) { if (w != e) memcpy(s->ev + ORA_EV * w, s->ev + ORA_EV * e, 8 * ORA_EV); ++w; }
                s->nev = w;
            }
            for (int c = 0; c < 3; ++c) { s->q[c * n + p] = gq[c * ng + ng - 1]; s->V[c * n + p] = gV[c * ng + ng - 1]; }
            s->R[p] = gR[ng - 1]; s->kind[p] = gkind[ng - 1];
            s->stat_groups++;
            if (ng > s->stat_maxgroup) s->stat_maxgroup = ng;
        }
        free(in); free(head); free(next);
    }
    free(idx); free(gm); free(grc); free(gq); free(gV);
    free(gR); free(gspin); free(gkind); free(m_pre); free(R_pre); free(spin_pre); free(kind_pre);
    return rcode;
}

/* End of a time step: ejections (L330-332) -- a body farther from the central mass than Rcut, or closer than RcutSun,
 * is reported and removed -- and the stop of the system (L378-384): when fewer than Nmin bodies are left, all of them
 * are removed.  Removed bodies are parked as the ghosts of the collisions are.  Event kinds: 2 = beyond Rcut,
 * 3 = inside RcutSun, 4 = removed because the system stopped. */
static void remove_body(ora_sys *s, int i, int kind_ev)
{
    int n = s->n;
    if (s->nev < s->evcap) {
        double *e = s->ev + ORA_EV * s->nev;
        memset(e, 0, 8 * ORA_EV);
        e[0] = (double)s->step_id; e[1] = kind_ev; e[2] = i; e[3] = -1; e[4] = s->m[i]; e[6] = s->R[i];
        for (int c = 0; c < 3; ++c) { e[8 + c] = s->q[c * n + i]; e[11 + c] = s->V[c * n + i]; e[21 + c] = s->spin[c * n + i]; }
    }
    s->nev++;
    double Rp = 1000.0 * (double)(i + 1);
    s->m[i] = 0.0; s->R[i] = 0.0; s->kind[i] = 2;
    s->spin[i] = s->spin[n + i] = s->spin[2 * n + i] = 0.0;
    s->q[i] = Rp; s->q[n + i] = 0.0; s->q[2 * n + i] = 0.0;
    s->V[i] = 0.0; s->V[n + i] = sqrt(s->G * s->m0 / Rp); s->V[2 * n + i] = 0.0;
}
static void end_of_step(ora_sys *s)
{
    int n = s->n;
    if (s->rcut > 0.0 || s->rcut_sun > 0.0)
        for (int i = 0; i < n; ++i) {
            if (s->kind[i] == 2) continue;
            double r2 = s->q[i] * s->q[i] + s->q[n + i] * s->q[n + i] + s->q[2 * n + i] * s->q[2 * n + i];
            if (s->rcut > 0.0 && r2 > s->rcut * s->rcut) remove_body(s, i, 2);
            else if (s->rcut_sun > 0.0 && r2 < s->rcut_sun * s->rcut_sun) remove_body(s, i, 3);
        }
    if (s->nmin > 0) {
        int left = 0;
        for (int i = 0; i < s->n_massive; ++i) left += s->kind[i] != 2;
        if (left < s->nmin && left > 0)
            for (int i = 0; i < n; ++i) if (s->kind[i] != 2) remove_body(s, i, 4);
    }
}

/* Second-order map S2(h), Eq. 7 (L100), in the order of the bullet list
 * L153-166, with the critical radii frozen [R-4]:
 *   B(h/2) + precheck, C(h/2), A(h) = Kepler drift + encounter search +
 *   grouping + BS on the groups, C(h/2), B(h/2). */
int ora_map_s2(ora_sys *s, double h)
{
    int rcode;
    rcode = kick(s, 0.5 * h, 1);                                   if (rcode) return rcode;
    if (!s->cull) { rcode = all_pairs(s);                           if (rcode) return rcode; }
    ora_sun_kick(s->n, s->n_massive, s->m0, s->m, s->V, s->q, 0.5 * h);
    memcpy(s->q0, s->q, 24 * (size_t)s->n); memcpy(s->V0, s->V, 24 * (size_t)s->n);
    rcode = ora_drift_all(s->n, s->G * s->m0, h, s->q, s->V, &s->stat_kepler_iters); if (rcode) return rcode;
    rcode = ora_confirm(s->n, s->q0, s->V0, s->q, s->V, s->rc, h, s->cand, s->n_cand,
                        s->enc, s->cap, &s->n_enc);                 if (rcode) return rcode;
    rcode = do_groups(s, h);                                        if (rcode) return rcode;
    ora_sun_kick(s->n, s->n_massive, s->m0, s->m, s->V, s->q, 0.5 * h);
    rcode = kick(s, 0.5 * h, 0);
    return rcode;
}

/* One full step of order 2, 4 or 6 (L146 "compute critical radii" once per time
 * step [R-4]; L168-170: Yoshida (1990) compositions of Eq. 7, sixth order =
 * "solutions A" [R-6]). */
int ora_yoshida(int order, double w[7])
{
    static const double w6[4] = {1.315186320683906, -1.17767998417887,
                                 0.235573213359357, 0.784513610477560}; /* w0..w3 */
    if (order == 2) { w[0] = 1.0; return 1; }
    if (order == 4) {
        double w1 = 1.0 / (2.0 - cbrt(2.0)), w0 = 1.0 - 2.0 * w1;
        w[0] = w1; w[1] = w0; w[2] = w1; return 3;
    }
    if (order == 6) {
        w[0] = w6[3]; w[1] = w6[2]; w[2] = w6[1]; w[3] = w6[0]; w[4] = w6[1]; w[5] = w6[2]; w[6] = w6[3];
        return 7;
    }
    return 0;
}
int ora_step(ora_sys *s, int64_t n_steps, double dt, int order)
{
    double w[7];
    int nw = ora_yoshida(order, w);
    if (nw == 0) return ORA_EINVAL;
    if (dt == 0.0) return ORA_EINVAL;
    for (int64_t t = 0; t < n_steps; ++t) {
        ora_rcrit(s->n, s->G, s->m0, s->n1, s->n2, dt, s->m, s->q, s->V, s->rc);
        for (int k = 0; k < nw; ++k) {
            int rcode = ora_map_s2(s, w[k] * dt);
            if (rcode) return rcode;
        }
        end_of_step(s);
        s->step_id++;
    }
    return ORA_OK;
}

/* accessors */
void ora_get_encounters(const ora_sys *s, int32_t *cand, int64_t *ncand, int32_t *enc,
                        int64_t *nenc, int32_t *label)
{
    *ncand = s->n_cand; *nenc = s->n_enc;
    int64_t nc = s->n_cand < s->cap ? s->n_cand : s->cap, ne = s->n_enc < s->cap ? s->n_enc : s->cap;
    if (cand) memcpy(cand, s->cand, 8 * (size_t)nc);
    if (enc) memcpy(enc, s->enc, 8 * (size_t)ne);
    if (label) memcpy(label, s->label, 4 * (size_t)s->n);
}
void ora_get_stats(const ora_sys *s, int64_t *out)
{
    out[0] = s->stat_kepler_iters; out[1] = s->stat_bs[0]; out[2] = s->stat_bs[1];
    out[3] = s->stat_force_evals; out[4] = s->stat_groups; out[5] = s->stat_maxgroup;
}
double ora_system_energy(const ora_sys *s, double *L)
{
    double E;
    ora_energy(s->n_massive, s->n, s->G, s->m0, s->m, s->q, s->V, NULL, &E, L, NULL);
    return E;
}
/* rc for the current state and step dt, plus the kick accelerations at it */
int ora_accel_now(ora_sys *s, double dt, double *a, double *rc)
{
    ora_rcrit(s->n, s->G, s->m0, s->n1, s->n2, dt, s->m, s->q, s->V, s->rc);
    int rcode = ora_accel(s->n, s->n_massive, s->G, s->m, s->q, s->rc, s->a, 1, s->cand, s->cap, &s->n_cand);
    memcpy(a, s->a, 24 * (size_t)s->n);
    if (rc) memcpy(rc, s->rc, 8 * (size_t)s->n);
    return rcode;
}
