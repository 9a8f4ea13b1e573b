// Kernels of the hybrid symplectic step, sm_100a.
// Each kernel states the operator it implements and the passage that defines it.
#define GENGA_KERNELS_CU 1
#include "kernels.cuh"
#include "bs_cluster.cuh"
#include "bs_warp.cuh"
#include "bs_small.cuh"

namespace genga {

// First statement of every kernel: let the next kernel of the stream be scheduled, then wait until the previous one has
// completed and its memory is visible (no-ops unless launched with programmatic stream serialization, api.cu launch_k).
__device__ __forceinline__ void pdl_sync()
{
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// the per-map counters: candidates, encounter pairs, groups, listed particles, the Bulirsch-Stoer queues and trace
__device__ __forceinline__ void reset_map_counters(const DevState &d)
{
    d.cnt[CI_NCAND] = 0; d.cnt[CI_NENC] = 0; d.cnt[CI_NGROUPS] = 0; d.cnt[CI_NTP] = 0; d.cnt[CI_NBIG] = 0;
    d.cnt[CI_QWARP] = 0; d.cnt[CI_QTP] = 0; d.cnt[CI_NTRACE] = 0; d.cnt[CI_NREDO] = 0; d.cnt[CI_NCAND_TP] = 0;
}
// one record per integrated group (genga_bs_trace): size, layout, accepted steps, rejected attempts, SM cycles
__device__ __forceinline__ void bs_trace(const DevState &d, int n, int layout, const int *nsteps, long long t0, int first)
{
    const int k = atomicAdd(&d.cnt[CI_NTRACE], 1);
    if (k < BS_TRACE_CAP) d.bstrace[k] = make_int4(n | (layout << 16), nsteps[0] | (nsteps[1] << 16), (int)(clock64() - t0), first);
}

// a group for k_bs_generic (collisions switched on): kind 0 massive group g, 1 particle p, 2 multi-system (system, member mask)
__device__ __forceinline__ void push_redo(const DevState &d, int kind, int id, int mask)
{
    const int k = atomicAdd(&d.cnt[CI_NREDO], 1);
    if (k < d.cap) d.redo[k] = make_int2((kind << 28) | id, mask);
    else atomicOr(&d.cnt[CI_STATUS], ERRBIT_CAPACITY);
}

// =====================================================================================
// Start of a map S2: forget the previous substep's lists.  Mode 1: clear the per-particle
// encounter masks of the particles listed last time.
__global__ void k_begin_map(DevState d)
{
    pdl_sync();
    int nprev = d.cnt[CI_NTP];
    if (d.mode == 1) {
        for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < nprev; k += gridDim.x * blockDim.x)
            d.tpmask[d.tplist[k] - d.nm] = 0u;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) d.cnt[CI_NTP_PREV] = nprev;
}
__global__ void k_reset_counters(DevState d)
{
    pdl_sync();
    if (threadIdx.x == 0) {
        reset_map_counters(d);
    }
}

// =====================================================================================
// Critical radius, Eq. 6 (L94-96): rc_i = max(n1 R_H,i , n2 |tau| v_i), v_i = |V_i| the body's
// own velocity (L96), R_H,i = a_i (m_i / 3 m0)^(1/3) with a_i from the vis-viva relation
// (r_i if unbound); test particles have R_H = 0.  Also stores 9 rc^2, the squared precheck
// distance (L142: "increasing the critical radius by a factor of three").
__device__ __forceinline__ double rcrit_of(double G, double m0, double n1, double n2, double tau,
                                           double x, double y, double z, double vx, double vy, double vz, double m)
{
    double r = sqrt(x * x + y * y + z * z);
    double v2 = vx * vx + vy * vy + vz * vz;
    double ainv = 2.0 / r - v2 / (G * m0);
    double a = ainv > 0.0 ? 1.0 / ainv : r;
    double rh = m > 0.0 ? a * cbrt(m / (3.0 * m0)) : 0.0;
    double rv = n2 * fabs(tau) * sqrt(v2);
    return fmax(n1 * rh, rv);
}
__global__ void k_rcrit(DevState d, double tau, int reset, int check)
{
    pdl_sync();
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (reset == 2) {                                     // mode 1 (ONE block): k_begin_map and k_reset_counters of the first map
        const int nprev = d.cnt[CI_NTP];
        for (int k = threadIdx.x; k < nprev; k += blockDim.x) d.tpmask[d.tplist[k] - d.nm] = 0u;
        __syncthreads();                                  // every thread has read the old count
        if (threadIdx.x == 0) d.cnt[CI_NTP_PREV] = nprev;
    }
    if (reset && i == 0) {                                // start of a step: forget the previous step's lists
        reset_map_counters(d);
    }
    // check & 2: the state did not come out of a step (set_state, an operator call): the packed j-tile of the kick is
    // written here too ; its padding up to a multiple of 128 sits far away and is massless
    const bool pack = (check & 2) && d.kb != nullptr;
    if (pack && i >= d.nm && i < d.npm) {
        reinterpret_cast<double4 *>(d.kb)[i] = make_double4(1e100, 1e100, 1e100, 0.0);
        d.hcw[i] = -1;
    }
    if (i >= d.ntot) return;
    double x = d.x[i], y = d.y[i], z = d.z[i], vx = d.vx[i], vy = d.vy[i], vz = d.vz[i], m = d.m[i];
    if (pack && i < d.nm) reinterpret_cast<double4 *>(d.kb)[i] = make_double4(x, y, z, d.G * m);
    double m0 = d.m0[system_of(d, i)];
    double n1 = d.n1, n2 = d.n2;
    if (d.mode == 2) { n1 = d.n12[2 * (i / d.nm)]; n2 = d.n12[2 * (i / d.nm) + 1]; }   // per system (L346-354)
    double rc = rcrit_of(d.G, m0, n1, n2, tau, x, y, z, vx, vy, vz, m);
    // S2': the hit masks of the previous closing kick cover r < 3.3 rc_old; they serve the coming opening kick only if
    // 3 rc_new <= 3.3 rc_old for every body
    if ((check & 1) && rc > KK_GROW * d.rc[i]) d.cnt[CI_S2PMISS] = 1;
    if (d.rcprev && i < d.nm) d.rcprev[i] = d.rc[i];           // mode 1: the particles' closing kick of the step that ends (k_tp_mid)
    d.rc[i] = rc;
    d.c9[i] = 9.0 * rc * rc;
    if (d.hcw && i < d.nm) d.hcw[i] = __double2hiint(KK_WIDE2 * rc * rc);
}

// =====================================================================================
// Kick, operator B (Eq. 2; L197, L238-264): V_i += h a_i, a_i = sum_j G m_j (q_j - q_i)/r^3
// W(r, rc_ij), and the prechecker (L142).  Massive bodies of one system, N <= 2048.
//
// Layout.  The paper gives every body i a thread block whose threads split the j loop and
// reduce in shared memory (Table 2).  Here one block per SM owns ni = ceil(N / #SM)
// <= 14 bodies i ("rows") and stages all bodies j once in shared memory (a 32-byte record
// x, y, z, G m_j per body, the high word of its precheck distance, its critical radius).
// A LANE owns two rows: their positions sit in registers and their sums never leave the lane,
// so the pair loop ends without any reduction over the 2048 partners, and every body j read
// from shared memory serves two pairs.  The 32 lanes of a warp are R row pairs x P phases;
// the lanes of one phase read the same body j (a multicast) and the P phases read P
// consecutive bodies.  14 rows = 8 + 4 + 2: warps 0-15 take rows 0-7 with P = 8, warps 16-23
// rows 8-11 with P = 16, warps 24-27 rows 12-13 with P = 32, and every warp covers 1/16, 1/8,
// 1/4 of the bodies j: all 28 warps (7 per SM sub-partition) run exactly ceil(N / 128) <= 16
// iterations of two pairs with all lanes busy.
//
// Per pair the fast path costs 16 FP64 issue slots: 3 subtractions, 3 for r^2, 7 for
// G m_j r^-3 from the MUFU.RSQ64H seed (rinv3_fast), 3 accumulating FMAs, and no branch.
// The precheck r^2 < 9 max(rc_i, rc_j)^2 is done on the HIGH WORDS of the doubles with
// integer compares (a superset of the exact test, off the FP64 pipe).  A pair that passes --
// the whole changeover zone r < rc_ij lies inside the precheck sphere, and so does the body
// itself -- gets weight 0 by clearing the seed and sets a bit in the lane's hit mask (two bits
// per iteration).  After its pair loop each warp lists its hits in a fixed order, evaluates
// them one per lane with the exact weight W = K - r dK/dr and the exact candidate test, and
// the row pair's first lane adds them in list order: no atomics on the sums, deterministic.  The row sums of the warps meet in shared memory and the block applies the
// kick to its own bodies: one launch, no partial sums in global memory.
__device__ __forceinline__ double kick_scale_exact(double r2, double rcij, double Gmj)
{
    // G m_j W(r, rc_ij) / r^3 with W of kick_weight(), arranged on the reciprocal seeds (a few ulp)
    double rinv = rsqrt_fast(r2);
    double r = r2 * rinv;
    double s3 = Gmj * (rinv * rinv) * rinv;
    double irc = rcp_fast(0.9 * rcij);
    double y = (r - 0.1 * rcij) * irc;
    if (!(y > 0.0)) return 0.0;
    if (y >= 1.0) return s3;
    double D = fma(2.0 * y, y - 1.0, 1.0);
    double iD = rcp_fast(D);
    double yD = y * iD;                                           // K = y yD
    double rdK = 2.0 * (1.0 - y) * (yD * iD) * (r * irc);
    return s3 * fma(y, yD, -rdK);
}

struct __align__(32) KickBody { double x, y, z, gm; };
struct KickHit { int code; int pad; double cx, cy, cz; };      // code = bit of the lane's hit mask << 8 | lane

struct KickSmem {
    KickBody body[KK_MAXN];                 // all bodies j, padded to a multiple of 64
    int hc[KK_MAXN];                        // high word of 9 rc_j^2 (-1 for padding)
    double rc[KK_MAXN];                     // critical radius (exact pass)
    KickHit list[KK_WARPS][32];             // per warp: hits of the current window of the exact pass
    double wsum[KK_WARPS][8][3];            // per warp: sums of its rows
    unsigned long long mbar[16];            // one mbarrier per slice of the j-tile (bulk copies)
};

// ---- TMA bulk copies (cp.async.bulk) and mbarriers: the j-tile of k_kick arrives slice by slice, a warp starts on its slice
// when that slice has landed instead of after a block-wide barrier over all 88 KB
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    unsigned ok;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!ok);
}

__global__ void __launch_bounds__(KK_THREADS, 1) k_kick(DevState d, double h, int record, int ni, double *aout, int to0, int s2p)
{
    pdl_sync();
    extern __shared__ __align__(32) unsigned char kk_raw[];
    KickSmem &S = *reinterpret_cast<KickSmem *>(kk_raw);
    const int N = d.nm, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int i0 = blockIdx.x * ni;
    const int nib = min(ni, N - i0);
    const int iters = (N + 127) >> 7;                  // iterations of every warp
    const int npad = iters << 7;

    // geometry of this warp: R row pairs x P phases, warp wi of its group, covering bodies [wi L, (wi + 1) L)
    const int logP = warp < 16 ? 3 : warp < 24 ? 4 : 5;
    const int wi = warp < 16 ? warp : warp < 24 ? warp - 16 : warp - 24;
    const int rowbase = warp < 16 ? 0 : warp < 24 ? 8 : 12;
    const int P = 1 << logP, phase = lane & (P - 1), rp = lane >> logP;
    const int ii = rowbase + 2 * rp, i = i0 + ii;
    const bool ok0 = ii < nib, ok1 = ii + 1 < nib;

    // stage the bodies j.  TMA path: the first 16 lanes issue, each for one slice of 8 * iters bodies (what one warp of the first group
    // covers), three bulk copies (records, precheck words, critical radii) that complete on the slice's mbarrier
    // S2' (L266-274): s2p & 2 = this is the opening kick of a step at the positions of the previous step's closing kick,
    // whose hit masks and far-pair sums are stored (s2p & 1 there); they hold as long as no critical radius grew past the
    // margin of the wide precheck (k_rcrit latches that in CI_S2PMISS, then the pair loop runs again).  With the stored
    // sums nothing is staged: the exact pass fetches the few bodies it needs from the packed records in L2.
    const bool stored = (s2p & 2) && d.cnt[CI_S2PMISS] == 0;
    const bool tma = !(s2p & 4) && !stored;
    const int slb = iters << 3;                         // bodies per slice; 16 slices = npad bodies
    if (stored) {
    } else if (tma) {
        if (tid < 16) {                                 // sixteen lanes, a slice each: the copies are issued side by side
            const int sl = tid;
            mbar_init(&S.mbar[sl], 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            mbar_expect_tx(&S.mbar[sl], (unsigned)slb * 32u);
            bulk_g2s(&S.body[sl * slb], d.kb + 4 * (size_t)sl * slb, (unsigned)slb * 32u, &S.mbar[sl]);
        }
        // the precheck words and critical radii (24 KB of the 88) through registers meanwhile; the block barrier below publishes them
        for (int j = tid; j < npad; j += KK_THREADS) { S.hc[j] = d.hcw[j]; S.rc[j] = d.rc[j]; }
    } else {
        // all loads of the (at most 3) rounds in flight together; the precheck word as k_rcrit forms it
        constexpr int ROUNDS = (KK_MAXN + KK_THREADS - 1) / KK_THREADS;
        double lx[ROUNDS], ly[ROUNDS], lz[ROUNDS], lm[ROUNDS], lr[ROUNDS];
#pragma unroll
        for (int q = 0; q < ROUNDS; ++q) {
            const int j = tid + q * KK_THREADS;
            const bool v = j < N;
            lx[q] = v ? d.x[j] : 1e100; ly[q] = v ? d.y[j] : 1e100; lz[q] = v ? d.z[j] : 1e100;
            lm[q] = v ? d.m[j] : 0.0; lr[q] = v ? d.rc[j] : -1.0;
        }
#pragma unroll
        for (int q = 0; q < ROUNDS; ++q) {
            const int j = tid + q * KK_THREADS;
            if (j < npad) {
                KickBody b;
                b.x = lx[q]; b.y = ly[q]; b.z = lz[q]; b.gm = d.G * lm[q];
                S.body[j] = b;
                S.rc[j] = lr[q];
                S.hc[j] = lr[q] >= 0.0 ? __double2hiint(KK_WIDE2 * lr[q] * lr[q]) : -1;
            }
        }
    }
    // a row that does not exist sits far away: it never passes the precheck and its sums are never read
    const double xi0 = ok0 ? d.x[i] : 1e150, yi0 = ok0 ? d.y[i] : 1e150, zi0 = ok0 ? d.z[i] : 1e150;
    const double xi1 = ok1 ? d.x[i + 1] : 1e150, yi1 = ok1 ? d.y[i + 1] : 1e150, zi1 = ok1 ? d.z[i + 1] : 1e150;
    const double rci0 = ok0 ? d.rc[i] : 0.0, rci1 = ok1 ? d.rc[i + 1] : 0.0;
    const int hci0 = ok0 ? __double2hiint(KK_WIDE2 * rci0 * rci0) : -1, hci1 = ok1 ? __double2hiint(KK_WIDE2 * rci1 * rci1) : -1;
    // the velocity component this thread will kick at the end: loaded now, off the critical path
    double vel0 = 0.0;
    if ((tid & 3) == 0 && (tid >> 2) < 3 * nib) {
        const int r = (tid >> 2) / 3, c = (tid >> 2) - 3 * r;
        vel0 = (c == 0 ? d.vx : c == 1 ? d.vy : d.vz)[i0 + r];
    }
    __syncthreads();

    if (tma) {                                          // my slices of the j-tile (the block barrier above published the mbarriers)
        const int s0 = wi << (logP - 3), ns = 1 << (logP - 3);
        for (int sl = s0; sl < s0 + ns; ++sl) mbar_wait(&S.mbar[sl], 0);
    }
    double ax0 = 0.0, ay0 = 0.0, az0 = 0.0, ax1 = 0.0, ay1 = 0.0, az1 = 0.0;
    unsigned hits = 0u;
    if ((s2p & 1) && blockIdx.x == 0 && tid == 0) d.cnt[CI_S2PMISS] = 0;      // read by the k_rcrit of the next step
    if (rowbase < nib) {                                // warp-uniform: the group has rows in this block
        const int L = iters << logP;
        if (stored) {
            hits = d.khits[(size_t)blockIdx.x * KK_THREADS + tid];
            if (phase == 0) {
                const double *f = d.kfar + ((size_t)blockIdx.x * KK_THREADS + tid) * 6;
                ax0 = f[0]; ay0 = f[1]; az0 = f[2]; ax1 = f[3]; ay1 = f[4]; az1 = f[5];
            }
        } else {
            const KickBody *pb = &S.body[wi * L + phase];
            const int *ph = &S.hc[wi * L + phase];
            unsigned bit = 1u;
#pragma unroll 2
            for (int t = 0; t < iters; ++t) {
                const KickBody bj = *pb;
                const int hcj = *ph;
                pb += P; ph += P;
                // both pairs in one straight-line block: their dependent chains overlap
                const double dx0 = bj.x - xi0, dy0 = bj.y - yi0, dz0 = bj.z - zi0;
                const double dx1 = bj.x - xi1, dy1 = bj.y - yi1, dz1 = bj.z - zi1;
                const double r20 = fma(dz0, dz0, fma(dy0, dy0, dx0 * dx0)), r21 = fma(dz1, dz1, fma(dy1, dy1, dx1 * dx1));
                const bool hit0 = __double2hiint(r20) <= max(hci0, hcj), hit1 = __double2hiint(r21) <= max(hci1, hcj);
                const int yh0 = __double2hiint(rsqrt_seed(r20)), yh1 = __double2hiint(rsqrt_seed(r21));
                // weight 0 for hits (and r2 == 0: the body itself): clear the seed
                const double y00 = __hiloint2double(hit0 ? 0 : yh0, 0), y01 = __hiloint2double(hit1 ? 0 : yh1, 0);
                const double u0 = y00 * y00, u1 = y01 * y01;
                const double e0 = fma(-r20, u0, 1.0), e1 = fma(-r21, u1, 1.0);
                const double w0 = y00 * u0, w1 = y01 * u1;
                const double p0 = fma(1.875, e0, 1.5), p1 = fma(1.875, e1, 1.5);
                const double s30 = bj.gm * fma(p0 * e0, w0, w0), s31 = bj.gm * fma(p1 * e1, w1, w1);   // G m_j y0^3 (1 + 3e/2 + 15 e^2/8)
                ax0 = fma(s30, dx0, ax0); ay0 = fma(s30, dy0, ay0); az0 = fma(s30, dz0, az0);
                ax1 = fma(s31, dx1, ax1); ay1 = fma(s31, dy1, ay1); az1 = fma(s31, dz1, az1);
                hits |= (hit0 ? bit : 0u) | (hit1 ? bit << 1 : 0u);     // bit 2 t + s: row s of this lane met body j of iteration t
                bit <<= 2;
            }
        }
        // the P phases of a row pair: every lane of the pair gets the sums of its two rows
        if (!stored) {
            for (int o = 1; o < P; o <<= 1) {
                ax0 += __shfl_xor_sync(0xffffffffu, ax0, o); ay0 += __shfl_xor_sync(0xffffffffu, ay0, o); az0 += __shfl_xor_sync(0xffffffffu, az0, o);
                ax1 += __shfl_xor_sync(0xffffffffu, ax1, o); ay1 += __shfl_xor_sync(0xffffffffu, ay1, o); az1 += __shfl_xor_sync(0xffffffffu, az1, o);
            }
            if (s2p & 1) {                              // keep the sums over the far pairs and the hit masks for the next opening kick
                d.khits[(size_t)blockIdx.x * KK_THREADS + tid] = hits;
                if (phase == 0) {
                    double *f = d.kfar + ((size_t)blockIdx.x * KK_THREADS + tid) * 6;
                    f[0] = ax0; f[1] = ay0; f[2] = az0; f[3] = ax1; f[4] = ay1; f[5] = az1;
                }
            }
        }
        __syncwarp();

        if (tma) {                                      // the exact pass reads any body: all slices
#pragma unroll 1
            for (int sl = 0; sl < 16; ++sl) mbar_wait(&S.mbar[sl], 0);
        }
        // ---- this warp's pairs inside the precheck sphere: exact weight, candidate list.
        // Lane l, bit 2 t + s of its hit mask: row rowbase + 2 (l >> logP) + s, body j = wi L + t P + (l & (P - 1)).  The hits are
        // listed in (lane, bit) order, 32 at a time; lane e evaluates entry e; the row pair's first lane adds its entries in list order.
        const unsigned word = hits;
        const int cnt = __popc(word);
        int inc = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int n = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += n; }
        const int total = __shfl_sync(0xffffffffu, inc, 31), off = inc - cnt;
        for (int base = 0; base < total; base += 32) {
            {
                unsigned wb = word;
                int e = off - base;
                while (wb) {
                    int b = __ffs(wb) - 1;
                    wb &= wb - 1;
                    if (e >= 0 && e < 32) S.list[warp][e].code = (b << 8) | lane;
                    ++e;
                }
            }
            __syncwarp();
            const int nwin = min(32, total - base);
            bool cand = false;
            int ci = 0, cj = 0;
            if (lane < nwin) {
                const int code = S.list[warp][lane].code, wd = code >> 8, b = code & 255;      // bit index, lane
                ci = i0 + rowbase + 2 * (b >> logP) + (wd & 1); cj = wi * L + ((wd >> 1) << logP) + (b & (P - 1));
                double cx = 0.0, cy = 0.0, cz = 0.0;
                if (cj != ci) {
                    KickBody bj, bi;
                    if (stored) {
                        const double4 rj = reinterpret_cast<const double4 *>(d.kb)[cj], ri = reinterpret_cast<const double4 *>(d.kb)[ci];
                        bj.x = rj.x; bj.y = rj.y; bj.z = rj.z; bj.gm = rj.w; bi.x = ri.x; bi.y = ri.y; bi.z = ri.z; bi.gm = ri.w;
                    } else { bj = S.body[cj]; bi = S.body[ci]; }
                    double dx = bj.x - bi.x, dy = bj.y - bi.y, dz = bj.z - bi.z;
                    double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                    const double rcij = stored ? fmax(d.rc[ci], d.rc[cj]) : fmax(S.rc[ci], S.rc[cj]);
                    double s3 = kick_scale_exact(r2, rcij, bj.gm);
                    cand = record && ci < cj && r2 < 9.0 * rcij * rcij;      // = max(9 rc_i^2, 9 rc_j^2) as k_rcrit rounds it
                    cx = s3 * dx; cy = s3 * dy; cz = s3 * dz;
                }
                S.list[warp][lane].cx = cx; S.list[warp][lane].cy = cy; S.list[warp][lane].cz = cz;
            }
            const unsigned cm = __ballot_sync(0xffffffffu, cand);
            if (cm) {
                int cb = 0;
                if (lane == 0) cb = atomicAdd(&d.cnt[CI_NCAND], __popc(cm));
                cb = __shfl_sync(0xffffffffu, cb, 0);
                if (cand) {
                    int idx = cb + __popc(cm & ((1u << lane) - 1u));
                    if (idx < d.cap) d.cand[idx] = make_int2(ci, cj);
                    else atomicOr(&d.cnt[CI_STATUS], ERRBIT_CAPACITY);
                }
            }
            __syncwarp();
            if (phase == 0) {
                for (int e = 0; e < nwin; ++e) {
                    const int code = S.list[warp][e].code;
                    if (((code & 255) >> logP) == rp) {
                        const double cx = S.list[warp][e].cx, cy = S.list[warp][e].cy, cz = S.list[warp][e].cz;
                        if ((code >> 8) & 1) { ax1 += cx; ay1 += cy; az1 += cz; } else { ax0 += cx; ay0 += cy; az0 += cz; }
                    }
                }
            }
            __syncwarp();
        }
        if (phase == 0) {
            S.wsum[warp][2 * rp][0] = ax0; S.wsum[warp][2 * rp][1] = ay0; S.wsum[warp][2 * rp][2] = az0;
            S.wsum[warp][2 * rp + 1][0] = ax1; S.wsum[warp][2 * rp + 1][1] = ay1; S.wsum[warp][2 * rp + 1][2] = az1;
        }
    }
    __syncthreads();
    // four lanes per sum (value v = 3 row + component): each adds a quarter of the row's warps, two shuffle levels join them
    if (tid < 4 * 3 * KK_NI + (32 - (4 * 3 * KK_NI) % 32) % 32) {
        const int v = tid >> 2, part = tid & 3;
        const bool live = v < 3 * nib;
        const int r = live ? v / 3 : 0, c = live ? v - 3 * r : 0;
        const int w0 = r < 8 ? 0 : r < 12 ? 16 : 24, nw = r < 8 ? 16 : r < 12 ? 8 : 4, rr = r < 8 ? r : r < 12 ? r - 8 : r - 12;
        double a = 0.0;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int w = part + 4 * k;
            if (live && w < nw) a += S.wsum[w0 + w][rr][c];
        }
        a += __shfl_xor_sync(0xffffffffu, a, 1);
        a += __shfl_xor_sync(0xffffffffu, a, 2);
        if (live && part == 0) {
            // to0: the kicked velocities go to the pre-drift arrays, which the fused Sun kick + drift (k_sun, hdrift != 0)
            // only reads -- no block of that launch may read a velocity array another block is overwriting
            double *vel = to0 ? (c == 0 ? d.vx0 : c == 1 ? d.vy0 : d.vz0) : (c == 0 ? d.vx : c == 1 ? d.vy : d.vz);
            vel[i0 + r] = fma(h, a, vel0);
            if (aout) aout[(size_t)c * d.ntot + i0 + r] = a;
        }
    }
}

size_t kick_smem_bytes() { return sizeof(KickSmem); }

// Kick of the test particles (L334-340): one thread per particle looping over the <= 32
// massive bodies, which sit in shared memory (broadcast reads).  Precheck against every
// massive body; candidate pairs are (massive j, particle i).
__global__ void __launch_bounds__(128) k_tp_kick(DevState d, double h, int record, double *aout)
{
    pdl_sync();
    __shared__ double sx[32], sy[32], sz[32], sgm[32], src[32];
    const int nm = d.nm;
    if (threadIdx.x < nm) {
        int j = threadIdx.x;
        sx[j] = d.x[j]; sy[j] = d.y[j]; sz[j] = d.z[j]; sgm[j] = d.G * d.m[j]; src[j] = d.rc[j];
    }
    __syncthreads();
    int i = nm + blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= d.ntot) return;
    double xi = d.x[i], yi = d.y[i], zi = d.z[i], rci = d.rc[i];
    double ax = 0, ay = 0, az = 0;
    for (int j = 0; j < nm; ++j) {
        double dx = sx[j] - xi, dy = sy[j] - yi, dz = sz[j] - zi;
        double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
        double rcij = fmax(rci, src[j]);
        double s3 = sgm[j] * rinv3_fast(r2);
        if (r2 < 9.0 * rcij * rcij) {
            double r = sqrt(r2);
            s3 = sgm[j] / (r2 * r) * kick_weight(r, rcij);
            if (record) {
                int idx = atomicAdd(&d.cnt[CI_NCAND], 1);
                if (idx < d.cap) d.cand[idx] = make_int2(j, i);
                else atomicOr(&d.cnt[CI_STATUS], ERRBIT_CAPACITY);
            }
        }
        ax = fma(s3, dx, ax); ay = fma(s3, dy, ay); az = fma(s3, dz, az);
    }
    if (aout) { aout[i] = ax; aout[d.ntot + i] = ay; aout[2 * (size_t)d.ntot + i] = az; }
    d.vx[i] = fma(h, ax, d.vx[i]); d.vy[i] = fma(h, ay, d.vy[i]); d.vz[i] = fma(h, az, d.vz[i]);
}

// Test particles, fused (L334-342): a particle meets only the <= 32 massive bodies and the star, so its
// whole half map is one pass over its 48 bytes of state instead of four kernels.
//   k_tp_front: [rc_i = n2 |tau| |V_i| at the start of a step (Eq. 6 with R_H = 0)]  B(h/2): kick by the
//               massive bodies + precheck, C(h/2): Sun kick, A(h): Kepler drift.  A particle that recorded a
//               candidate keeps its state before the drift (Eq. 10 and Bulirsch-Stoer need it).
//   k_tp_back : C(h/2), B(h/2) at the end of the map (no precheck).
// psum must hold sum m V of the massive bodies after their own kick (front) / after Bulirsch-Stoer (back);
// the massive bodies must not have been shifted yet (front) / must have been shifted (back): B only sees
// differences of positions, which a common shift leaves alone.
struct TpMassive { double x[32], y[32], z[32], gm[32], rc[32]; int hc[32]; };
__device__ __forceinline__ void tp_load_massive(const DevState &d, TpMassive &M, const double *px, const double *py, const double *pz)
{
    if (threadIdx.x < d.nm) {
        int j = threadIdx.x;
        M.x[j] = px[j]; M.y[j] = py[j]; M.z[j] = pz[j]; M.gm[j] = d.G * d.m[j]; M.rc[j] = d.rc[j];
        M.hc[j] = __double2hiint(9.0 * M.rc[j] * M.rc[j]);
    }
    __syncthreads();
}
// acceleration of a particle at (xi, yi, zi) by the massive bodies; returns the mask of the massive bodies inside the
// precheck sphere (the particle's candidates, L142)
__device__ __forceinline__ unsigned tp_accel(const DevState &d, const TpMassive &M, double xi, double yi, double zi, double rci,
                                             double &ax, double &ay, double &az)
{
    unsigned cmask = 0u;
    ax = ay = az = 0.0;
    const int nm = d.nm;
    const int hci = __double2hiint(9.0 * rci * rci);            // precheck on the high words (a superset, off the FP64 pipe)
    for (int j = 0; j < nm; ++j) {
        double dx = M.x[j] - xi, dy = M.y[j] - yi, dz = M.z[j] - zi;
        double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
        double s3 = M.gm[j] * rinv3_fast(r2);
        if (__double2hiint(r2) <= max(hci, M.hc[j])) {
            const double rcij = fmax(rci, M.rc[j]);
            if (r2 < 9.0 * rcij * rcij) cmask |= 1u << j;
            if (r2 < rcij * rcij) {                             // inside the changeover zone: exact weight (W = 1 outside)
                double r = sqrt(r2);
                s3 = M.gm[j] / (r2 * r) * kick_weight(r, rcij);
            }
        }
        ax = fma(s3, dx, ax); ay = fma(s3, dy, ay); az = fma(s3, dz, az);
    }
    return cmask;
}
// The massive bodies have been kicked, Sun-kicked and drifted before this launch (k_tpm_kick, k_drift): x0.. hold them
// after the Sun kick, x.. after the drift.  The particle takes its Sun kick FIRST and its kick against the shifted massive
// bodies (B and C commute exactly: B only sees differences of positions, R-11), drifts, and tests its candidates by the
// Hermite minimum (Eq. 10-12) right here, from registers and shared memory: no candidate list, no gather, and the state
// before the drift is stored only for the few particles that do have an encounter.
struct TpMassive2 { double x1[32], y1[32], z1[32], vx0[32], vy0[32], vz0[32], vx1[32], vy1[32], vz1[32]; };
// Kepler drift of a particle, then its candidates tested by the Hermite minimum (Eq. 10-12) from registers and shared
// memory; the particle's state is written, the state before the drift only if it has an encounter.
__device__ __forceinline__ void tp_drift_confirm(const DevState &d, const TpMassive &M, const TpMassive2 &M2, const int i, const bool live,
                                                 const double h, const unsigned cmask, const double rci,
                                                 double x, double y, double z, double vx, double vy, double vz)
{
    const double x0 = x, y0 = y, z0 = z, vx0 = vx, vy0 = vy, vz0 = vz;
    if (live && !kepler_drift(d.G * d.m0[0], h, x, y, z, vx, vy, vz)) atomicOr(&d.cnt[CI_STATUS], ERRBIT_KEPLER);
    // candidates of this warp: one atomic
    {
        int nc = __popc(cmask);
        for (int o = 16; o > 0; o >>= 1) nc += __shfl_xor_sync(0xffffffffu, nc, o);
        if ((threadIdx.x & 31) == 0 && nc) atomicAdd(&d.cnt[CI_NCAND_TP], nc);
    }
    if (!live) return;
    unsigned emask = 0u;
    for (unsigned cm = cmask; cm; cm &= cm - 1) {
        const int j = __ffs(cm) - 1;
        double dx = x0 - M.x[j], dy = y0 - M.y[j], dz = z0 - M.z[j];
        double dvx = vx0 - M2.vx0[j], dvy = vy0 - M2.vy0[j], dvz = vz0 - M2.vz0[j];
        const double P0 = dx * dx + dy * dy + dz * dz, Pd0 = 2.0 * (dx * dvx + dy * dvy + dz * dvz);
        dx = x - M2.x1[j]; dy = y - M2.y1[j]; dz = z - M2.z1[j];
        dvx = vx - M2.vx1[j]; dvy = vy - M2.vy1[j]; dvz = vz - M2.vz1[j];
        const double P1 = dx * dx + dy * dy + dz * dz, Pd1 = 2.0 * (dx * dvx + dy * dvy + dz * dvz);
        const double rcij = fmax(rci, M.rc[j]);
        // a rigorous lower bound of the interpolant first (bs.cuh pair_collides): most candidates sit between rc and 3 rc
        if (pair_collides(P0, P1, Pd0, Pd1, h, rcij)) {
            emask |= 1u << j;
            const int idx = atomicAdd(&d.cnt[CI_NENC], 1);
            if (idx < d.cap) d.enc[idx] = make_int2(j, i);
            else atomicOr(&d.cnt[CI_STATUS], ERRBIT_CAPACITY);
        }
    }
    if (emask) {                                                // Bulirsch-Stoer needs the state before the drift
        d.x0[i] = x0; d.y0[i] = y0; d.z0[i] = z0; d.vx0[i] = vx0; d.vy0[i] = vy0; d.vz0[i] = vz0;
        d.tpmask[i - d.nm] = emask;
        d.tplist[atomicAdd(&d.cnt[CI_NTP], 1)] = i;
    }
    d.x[i] = x; d.y[i] = y; d.z[i] = z; d.vx[i] = vx; d.vy[i] = vy; d.vz[i] = vz;
}
__global__ void __launch_bounds__(128) k_tp_front(DevState d, double h, double tau, int first)
{
    pdl_sync();
    __shared__ TpMassive M;
    __shared__ TpMassive2 M2;
    const int i = d.nm + blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = i < d.ntot;
    // the particle's own loads go out before the block waits for the massive bodies: one memory round trip
    double x = 0.0, y = 0.0, z = 0.0, vx = 0.0, vy = 0.0, vz = 0.0, rci = 0.0;
    if (live) {
        x = d.x[i]; y = d.y[i]; z = d.z[i]; vx = d.vx[i]; vy = d.vy[i]; vz = d.vz[i];
        if (!first) rci = d.rc[i];
    }
    if (threadIdx.x < d.nm) {
        const int j = threadIdx.x;
        M2.x1[j] = d.x[j]; M2.y1[j] = d.y[j]; M2.z1[j] = d.z[j];
        M2.vx0[j] = d.vx0[j]; M2.vy0[j] = d.vy0[j]; M2.vz0[j] = d.vz0[j];
        M2.vx1[j] = d.vx[j]; M2.vy1[j] = d.vy[j]; M2.vz1[j] = d.vz[j];
    }
    tp_load_massive(d, M, d.x0, d.y0, d.z0);
    if (first && live) {
        rci = fmax(d.n1 * 0.0, d.n2 * fabs(tau) * sqrt(vx * vx + vy * vy + vz * vz));
        d.rc[i] = rci;
    }
    const double hh = 0.5 * h, g = hh / d.m0[0];
    x = fma(g, d.psum[0], x); y = fma(g, d.psum[1], y); z = fma(g, d.psum[2], z);
    double ax, ay, az;
    const unsigned cmask = live ? tp_accel(d, M, x, y, z, rci, ax, ay, az) : 0u;
    if (live) { vx = fma(hh, ax, vx); vy = fma(hh, ay, vy); vz = fma(hh, az, vz); }
    tp_drift_confirm(d, M, M2, i, live, h, cmask, rci, x, y, z, vx, vy, vz);
}
// Closing half of a map and opening half of the next one in ONE pass over the particle (the positions are the same):
//   C(hA/2) B(hA/2) | [new step: rc_i = n2 |tau| |V_i|] B(hB/2) C(hB/2) A(hB) + encounter search.
// The massive bodies have already gone through the same (k_tpm_kick closing, k_rcrit, k_tpm_kick opening, k_drift): x0..
// hold them after BOTH Sun kicks, so the particle takes both shifts first and kicks against x0 (B and C commute, R-11);
// psum + 4 = sum m V of the closing Sun kick, psum = of the opening one; rcprev = the massive bodies' critical radii of
// the step that ends (newstep).  Within a step (newstep = 0) the two kicks have the same weights: one evaluation.
__global__ void __launch_bounds__(128) k_tp_mid(DevState d, double hA, double hB, double tau, int newstep)
{
    pdl_sync();
    __shared__ TpMassive M;
    __shared__ TpMassive2 M2;
    __shared__ double rcold[32];
    __shared__ int hcold[32];
    const int i = d.nm + blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = i < d.ntot;
    double x = 0.0, y = 0.0, z = 0.0, vx = 0.0, vy = 0.0, vz = 0.0, rci = 0.0;
    if (live) { x = d.x[i]; y = d.y[i]; z = d.z[i]; vx = d.vx[i]; vy = d.vy[i]; vz = d.vz[i]; rci = d.rc[i]; }
    if (threadIdx.x < d.nm) {
        const int j = threadIdx.x;
        M2.x1[j] = d.x[j]; M2.y1[j] = d.y[j]; M2.z1[j] = d.z[j];
        M2.vx0[j] = d.vx0[j]; M2.vy0[j] = d.vy0[j]; M2.vz0[j] = d.vz0[j];
        M2.vx1[j] = d.vx[j]; M2.vy1[j] = d.vy[j]; M2.vz1[j] = d.vz[j];
        const double ro = newstep ? d.rcprev[j] : d.rc[j];
        rcold[j] = ro; hcold[j] = __double2hiint(9.0 * ro * ro);
    }
    tp_load_massive(d, M, d.x0, d.y0, d.z0);
    const double gA = 0.5 * hA / d.m0[0], gB = 0.5 * hB / d.m0[0];
    x = fma(gA, d.psum[4], x); y = fma(gA, d.psum[5], y); z = fma(gA, d.psum[6], z);
    x = fma(gB, d.psum[0], x); y = fma(gB, d.psum[1], y); z = fma(gB, d.psum[2], z);
    double ax, ay, az;
    unsigned cmask = 0u;
    if (newstep) {
        // closing kick with the critical radii of the step that ends
        if (live) {
            ax = ay = az = 0.0;
            const int hci = __double2hiint(9.0 * rci * rci);
            for (int j = 0; j < d.nm; ++j) {
                double dx = M.x[j] - x, dy = M.y[j] - y, dz = M.z[j] - z;
                double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                double s3 = M.gm[j] * rinv3_fast(r2);
                if (__double2hiint(r2) <= max(hci, hcold[j])) {
                    const double rcij = fmax(rci, rcold[j]);
                    if (r2 < rcij * rcij) {
                        double r = sqrt(r2);
                        s3 = M.gm[j] / (r2 * r) * kick_weight(r, rcij);
                    }
                }
                ax = fma(s3, dx, ax); ay = fma(s3, dy, ay); az = fma(s3, dz, az);
            }
            vx = fma(0.5 * hA, ax, vx); vy = fma(0.5 * hA, ay, vy); vz = fma(0.5 * hA, az, vz);
            rci = fmax(d.n1 * 0.0, d.n2 * fabs(tau) * sqrt(vx * vx + vy * vy + vz * vz));
            d.rc[i] = rci;
            cmask = tp_accel(d, M, x, y, z, rci, ax, ay, az);
            vx = fma(0.5 * hB, ax, vx); vy = fma(0.5 * hB, ay, vy); vz = fma(0.5 * hB, az, vz);
        }
    } else if (live) {
        cmask = tp_accel(d, M, x, y, z, rci, ax, ay, az);
        vx = fma(0.5 * hA, ax, vx); vy = fma(0.5 * hA, ay, vy); vz = fma(0.5 * hA, az, vz);     // two kicks, as k_tp_back and k_tp_front apply them
        vx = fma(0.5 * hB, ax, vx); vy = fma(0.5 * hB, ay, vy); vz = fma(0.5 * hB, az, vz);
    }
    tp_drift_confirm(d, M, M2, i, live, hB, cmask, rci, x, y, z, vx, vy, vz);
}
__global__ void __launch_bounds__(128) k_tp_back(DevState d, double h)
{
    pdl_sync();
    __shared__ TpMassive M;
    const int i = d.nm + blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = i < d.ntot;
    double x = 0.0, y = 0.0, z = 0.0, vx = 0.0, vy = 0.0, vz = 0.0, rci = 0.0;
    if (live) { x = d.x[i]; y = d.y[i]; z = d.z[i]; vx = d.vx[i]; vy = d.vy[i]; vz = d.vz[i]; rci = d.rc[i]; }
    tp_load_massive(d, M, d.x, d.y, d.z);
    if (!live) return;
    const double hh = 0.5 * h, g = hh / d.m0[0];
    x = fma(g, d.psum[4], x); y = fma(g, d.psum[5], y); z = fma(g, d.psum[6], z);      // the closing k_tpm_kick's sum
    double ax, ay, az;
    tp_accel(d, M, x, y, z, rci, ax, ay, az);
    d.x[i] = x; d.y[i] = y; d.z[i] = z;
    d.vx[i] = fma(hh, ax, vx); d.vy[i] = fma(hh, ay, vy); d.vz[i] = fma(hh, az, vz);
}

// Kick in multi-system mode (L368-370): one thread per body, partners = the bodies of its own system
// (contiguous, body = system * nm + k).  A block takes 128 / nm whole systems and stages their bodies in shared
// memory once (coalesced), so the partner loop reads shared memory (the lanes of a system read the same address).
__global__ void __launch_bounds__(128) k_kick_multi(DevState d, double h, int record, double *aout)
{
    pdl_sync();
    __shared__ double sx[128], sy[128], sz[128], sgm[128], src[128];
    const int nm = d.nm, spb = 128 / nm, t = threadIdx.x;
    const int i = blockIdx.x * spb * nm + t;
    const bool live = t < spb * nm && i < d.ntot;
    double xi = 0.0, yi = 0.0, zi = 0.0, rci = 0.0, vx = 0.0, vy = 0.0, vz = 0.0;
    if (live) {
        xi = d.x[i]; yi = d.y[i]; zi = d.z[i]; rci = d.rc[i];
        vx = d.vx[i]; vy = d.vy[i]; vz = d.vz[i];
        sx[t] = xi; sy[t] = yi; sz[t] = zi; src[t] = rci; sgm[t] = d.G * d.m[i];
    }
    __syncthreads();
    if (!live) return;
    const int sb = (t / nm) * nm;
    double ax = 0, ay = 0, az = 0;
    for (int k = 0; k < nm; ++k) {
        const int jt = sb + k;
        if (jt == t) continue;
        double dx = sx[jt] - xi, dy = sy[jt] - yi, dz = sz[jt] - zi;
        double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
        double rcij = fmax(rci, src[jt]);
        double gm = sgm[jt];
        double s3 = gm * rinv3_fast(r2);
        if (r2 < 9.0 * rcij * rcij) {
            if (r2 < rcij * rcij) {                             // W = 1 outside the changeover zone
                double r = sqrt(r2);
                s3 = gm / (r2 * r) * kick_weight(r, rcij);
            }
            const int j = i - t + jt;
            if (record && i < j) {
                int idx = atomicAdd(&d.cnt[CI_NCAND], 1);
                if (idx < d.cap) d.cand[idx] = make_int2(i, j);
                else atomicOr(&d.cnt[CI_STATUS], ERRBIT_CAPACITY);
            }
        }
        ax = fma(s3, dx, ax); ay = fma(s3, dy, ay); az = fma(s3, dz, az);
    }
    if (aout) { aout[i] = ax; aout[d.ntot + i] = ay; aout[2 * (size_t)d.ntot + i] = az; }
    d.vx[i] = fma(h, ax, vx); d.vy[i] = fma(h, ay, vy); d.vz[i] = fma(h, az, vz);
}

// The massive bodies of the test-particle mode (nm <= 32, L188): kick, momentum sum and Sun kick of one half map in ONE
// warp (body = lane).  fshift == 0, opening half: kick, then s = sum m V for the particles' and the massive bodies' Sun kick
// (k_tp_front, k_drift).  fshift != 0, closing half: s from the velocities as they are, q += fshift s / m0, then the kick at
// the shifted positions.  Same pair arithmetic as k_kick_multi, same sum order as k_momentum with 32 threads.
__global__ void __launch_bounds__(32) k_tpm_kick(DevState d, double h, int record, double fshift, int slot)
{
    pdl_sync();
    __shared__ double sx[32], sy[32], sz[32], sgm[32], src[32];
    const int t = threadIdx.x, nm = d.nm;
    const bool live = t < nm;
    double xi = 0.0, yi = 0.0, zi = 0.0, rci = 0.0, vx = 0.0, vy = 0.0, vz = 0.0, m = 0.0;
    if (live) {
        xi = d.x[t]; yi = d.y[t]; zi = d.z[t]; rci = d.rc[t];
        vx = d.vx[t]; vy = d.vy[t]; vz = d.vz[t]; m = d.m[t];
    }
    auto momentum = [&](double &s0, double &s1, double &s2) {
        s0 = m * vx; s1 = m * vy; s2 = m * vz;
        double s3 = m;
        for (int o = 16; o > 0; o >>= 1) {
            s0 += __shfl_xor_sync(0xffffffffu, s0, o); s1 += __shfl_xor_sync(0xffffffffu, s1, o);
            s2 += __shfl_xor_sync(0xffffffffu, s2, o); s3 += __shfl_xor_sync(0xffffffffu, s3, o);
        }
        if (t == 0) { d.psum[4 * slot] = s0; d.psum[4 * slot + 1] = s1; d.psum[4 * slot + 2] = s2; d.psum[4 * slot + 3] = s3; }
    };
    if (fshift != 0.0) {
        double s0, s1, s2;
        momentum(s0, s1, s2);
        const double g = fshift / d.m0[0];
        xi = fma(g, s0, xi); yi = fma(g, s1, yi); zi = fma(g, s2, zi);
        if (live) { d.x[t] = xi; d.y[t] = yi; d.z[t] = zi; }
    }
    sx[t] = xi; sy[t] = yi; sz[t] = zi; src[t] = rci; sgm[t] = d.G * m;
    __syncwarp();
    double ax = 0, ay = 0, az = 0;
    if (live) {
        for (int j = 0; j < nm; ++j) {
            if (j == t) continue;
            double dx = sx[j] - xi, dy = sy[j] - yi, dz = sz[j] - zi;
            double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            double rcij = fmax(rci, src[j]);
            double gm = sgm[j];
            double s3 = gm * rinv3_fast(r2);
            if (r2 < 9.0 * rcij * rcij) {
                if (r2 < rcij * rcij) {                             // W = 1 outside the changeover zone
                    double r = sqrt(r2);
                    s3 = gm / (r2 * r) * kick_weight(r, rcij);
                }
                if (record && t < j) {
                    int idx = atomicAdd(&d.cnt[CI_NCAND], 1);
                    if (idx < d.cap) d.cand[idx] = make_int2(t, j);
                    else atomicOr(&d.cnt[CI_STATUS], ERRBIT_CAPACITY);
                }
            }
            ax = fma(s3, dx, ax); ay = fma(s3, dy, ay); az = fma(s3, dz, az);
        }
        vx = fma(h, ax, vx); vy = fma(h, ay, vy); vz = fma(h, az, vz);
        d.vx[t] = vx; d.vy[t] = vy; d.vz[t] = vz;
    }
    if (fshift == 0.0) {
        double s0, s1, s2;
        momentum(s0, s1, s2);
    }
}

// Massive mode with N <= 32 (the paper's small-N regime, L427-433, where a step is launch latency): ONE warp, body = lane,
// runs a whole half map per launch.  Pair arithmetic as k_kick_multi, critical radius as k_rcrit, Sun kick and drift as k_sun.
__device__ __forceinline__ void tiny_reset(const DevState &d)
{
    reset_map_counters(d);
}
struct TinySmem { double x[32], y[32], z[32], gm[32], rc[32]; };
__device__ __forceinline__ void tiny_kick(const DevState &d, TinySmem &S, int t, bool live, double h, int record,
                                          double xi, double yi, double zi, double rci, double m,
                                          double &vx, double &vy, double &vz)
{
    S.x[t] = xi; S.y[t] = yi; S.z[t] = zi; S.rc[t] = rci; S.gm[t] = d.G * m;
    __syncwarp();
    if (live) {
        double ax = 0, ay = 0, az = 0;
        for (int j = 0; j < d.nm; ++j) {
            if (j == t) continue;
            double dx = S.x[j] - xi, dy = S.y[j] - yi, dz = S.z[j] - zi;
            double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            double rcij = fmax(rci, S.rc[j]);
            double gm = S.gm[j];
            double s3 = gm * rinv3_fast(r2);
            if (r2 < 9.0 * rcij * rcij) {
                if (r2 < rcij * rcij) {                             // W = 1 outside the changeover zone
                    double r = sqrt(r2);
                    s3 = gm / (r2 * r) * kick_weight(r, rcij);
                }
                if (record && t < j) {
                    int idx = atomicAdd(&d.cnt[CI_NCAND], 1);
                    if (idx < d.cap) d.cand[idx] = make_int2(t, j);
                    else atomicOr(&d.cnt[CI_STATUS], ERRBIT_CAPACITY);
                }
            }
            ax = fma(s3, dx, ax); ay = fma(s3, dy, ay); az = fma(s3, dz, az);
        }
        vx = fma(h, ax, vx); vy = fma(h, ay, vy); vz = fma(h, az, vz);
    }
    __syncwarp();
}
__device__ __forceinline__ void tiny_momentum(double m, double vx, double vy, double vz, double &s0, double &s1, double &s2)
{
    s0 = m * vx; s1 = m * vy; s2 = m * vz;
    for (int o = 16; o > 0; o >>= 1) {
        s0 += __shfl_xor_sync(0xffffffffu, s0, o); s1 += __shfl_xor_sync(0xffffffffu, s1, o); s2 += __shfl_xor_sync(0xffffffffu, s2, o);
    }
}
// opening half of a map: [critical radii and counter reset at the first map of a step] [kick B(hk), recording the candidates]
// Sun kick C(h/2), Kepler drift A(h)
__global__ void __launch_bounds__(32) k_tiny_front(DevState d, double h, double tau, int first, double hk)
{
    pdl_sync();
    __shared__ TinySmem S;
    const int t = threadIdx.x;
    const bool live = t < d.nm;
    double x = 0.0, y = 0.0, z = 0.0, vx = 0.0, vy = 0.0, vz = 0.0, m = 0.0, rc = 0.0;
    const double m0 = d.m0[0];
    if (live) { x = d.x[t]; y = d.y[t]; z = d.z[t]; vx = d.vx[t]; vy = d.vy[t]; vz = d.vz[t]; m = d.m[t]; }
    if (first) {
        if (t == 0) tiny_reset(d);
        if (live) { rc = rcrit_of(d.G, m0, d.n1, d.n2, tau, x, y, z, vx, vy, vz, m); d.rc[t] = rc; d.c9[t] = 9.0 * rc * rc; }
        __syncwarp();
    } else if (live) rc = d.rc[t];
    if (hk != 0.0) tiny_kick(d, S, t, live, hk, 1, x, y, z, rc, m, vx, vy, vz);
    double s0, s1, s2;
    tiny_momentum(m, vx, vy, vz, s0, s1, s2);
    __shared__ double Q[12][32], src[32];                     // state before and after the drift, critical radii
    if (live) {
        const double g = 0.5 * h / m0;
        x = fma(g, s0, x); y = fma(g, s1, y); z = fma(g, s2, z);
        d.x0[t] = x; d.y0[t] = y; d.z0[t] = z; d.vx0[t] = vx; d.vy0[t] = vy; d.vz0[t] = vz;
        Q[0][t] = x; Q[1][t] = y; Q[2][t] = z; Q[3][t] = vx; Q[4][t] = vy; Q[5][t] = vz;
        if (!kepler_drift(d.G * m0, h, x, y, z, vx, vy, vz)) atomicOr(&d.cnt[CI_STATUS], ERRBIT_KEPLER);
        d.x[t] = x; d.y[t] = y; d.z[t] = z; d.vx[t] = vx; d.vy[t] = vy; d.vz[t] = vz;
        Q[6][t] = x; Q[7][t] = y; Q[8][t] = z; Q[9][t] = vx; Q[10][t] = vy; Q[11][t] = vz;
        src[t] = rc;
    }
    __syncwarp();
    // encounter search over the candidates (k_confirm's arithmetic; the candidates come from this launch's kick or from
    // the merged kick of the previous map's k_tiny_back)
    const int nc = min(atomicAdd(&d.cnt[CI_NCAND], 0), (int)d.cap);
    for (int e = t; e < nc; e += 32) {
        const int2 p = __ldcg(&d.cand[e]);
        const int i = p.x, j = p.y;
        double dx = Q[0][j] - Q[0][i], dy = Q[1][j] - Q[1][i], dz = Q[2][j] - Q[2][i];
        double dvx = Q[3][j] - Q[3][i], dvy = Q[4][j] - Q[4][i], dvz = Q[5][j] - Q[5][i];
        double P0 = dx * dx + dy * dy + dz * dz, Pd0 = 2.0 * (dx * dvx + dy * dvy + dz * dvz);
        dx = Q[6][j] - Q[6][i]; dy = Q[7][j] - Q[7][i]; dz = Q[8][j] - Q[8][i];
        dvx = Q[9][j] - Q[9][i]; dvy = Q[10][j] - Q[10][i]; dvz = Q[11][j] - Q[11][i];
        double P1 = dx * dx + dy * dy + dz * dz, Pd1 = 2.0 * (dx * dvx + dy * dvy + dz * dvz);
        double rcij = fmax(src[i], src[j]);
        double D = hermite_min(P0, P1, Pd0, Pd1, h);
        if (D < rcij * rcij) {
            int idx = atomicAdd(&d.cnt[CI_NENC], 1);
            if (idx < d.cap) d.enc[idx] = p;
            else atomicOr(&d.cnt[CI_STATUS], ERRBIT_CAPACITY);
        }
    }
}
// closing half of a map: Sun kick C(h/2) [counter reset: the map is over], kick B(hk) [recording the next map's candidates]
__global__ void __launch_bounds__(32) k_tiny_back(DevState d, double h, double hk, int record, int reset)
{
    pdl_sync();
    __shared__ TinySmem S;
    const int t = threadIdx.x;
    const bool live = t < d.nm;
    double x = 0.0, y = 0.0, z = 0.0, vx = 0.0, vy = 0.0, vz = 0.0, m = 0.0, rc = 0.0;
    if (live) { x = d.x[t]; y = d.y[t]; z = d.z[t]; vx = d.vx[t]; vy = d.vy[t]; vz = d.vz[t]; m = d.m[t]; rc = d.rc[t]; }
    if (reset) {
        if (t == 0) tiny_reset(d);
        __syncwarp();
    }
    double s0, s1, s2;
    tiny_momentum(m, vx, vy, vz, s0, s1, s2);
    const double g = 0.5 * h / d.m0[0];
    x = fma(g, s0, x); y = fma(g, s1, y); z = fma(g, s2, z);
    tiny_kick(d, S, t, live, hk, record, x, y, z, rc, m, vx, vy, vz);
    if (!live) return;
    d.x[t] = x; d.y[t] = y; d.z[t] = z; d.vx[t] = vx; d.vy[t] = vy; d.vz[t] = vz;
}

// Multi-system mode, half maps in one launch (a block holds whole systems, so nothing crosses blocks): the pair loop of
// k_kick_multi, the momentum sum, Sun kick and drift of k_sun with the same arithmetic in the same order.
struct MultiSmem { double x[128], y[128], z[128], gm[128], rc[128], m[128], vx[128], vy[128], vz[128]; };
__device__ __forceinline__ void multi_pairs(const DevState &d, const MultiSmem &S, int t, int i, int sb, int record,
                                            double xi, double yi, double zi, double rci, double &ax, double &ay, double &az)
{
    ax = ay = az = 0.0;
    for (int k = 0; k < d.nm; ++k) {
        const int jt = sb + k;
        if (jt == t) continue;
        double dx = S.x[jt] - xi, dy = S.y[jt] - yi, dz = S.z[jt] - zi;
        double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
        double rcij = fmax(rci, S.rc[jt]);
        double gm = S.gm[jt];
        double s3 = gm * rinv3_fast(r2);
        if (r2 < 9.0 * rcij * rcij) {
            if (r2 < rcij * rcij) {                             // W = 1 outside the changeover zone
                double r = sqrt(r2);
                s3 = gm / (r2 * r) * kick_weight(r, rcij);
            }
            const int j = i - t + jt;
            if (record && i < j) {
                int idx = atomicAdd(&d.cnt[CI_NCAND], 1);
                if (idx < d.cap) d.cand[idx] = make_int2(i, j);
                else atomicOr(&d.cnt[CI_STATUS], ERRBIT_CAPACITY);
            }
        }
        ax = fma(s3, dx, ax); ay = fma(s3, dy, ay); az = fma(s3, dz, az);
    }
}
// opening half: [kick B(hk), recording the candidates] Sun kick C(h/2), drift A(h); labels reset for the map's grouping
__global__ void __launch_bounds__(128) k_multi_front(DevState d, double h, double hk)
{
    pdl_sync();
    __shared__ MultiSmem S;
    const int nm = d.nm, spb = 128 / nm, t = threadIdx.x;
    const int i = blockIdx.x * spb * nm + t;
    const bool live = t < spb * nm && i < d.ntot;
    double x = 0.0, y = 0.0, z = 0.0, rc = 0.0, vx = 0.0, vy = 0.0, vz = 0.0, m = 0.0;
    if (live) {
        x = d.x[i]; y = d.y[i]; z = d.z[i]; rc = d.rc[i]; vx = d.vx[i]; vy = d.vy[i]; vz = d.vz[i]; m = d.m[i];
        d.label[i] = i;
        S.x[t] = x; S.y[t] = y; S.z[t] = z; S.rc[t] = rc; S.gm[t] = d.G * m; S.m[t] = m;
    }
    __syncthreads();
    const int sb = (t / nm) * nm;
    if (live && hk != 0.0) {
        double ax, ay, az;
        multi_pairs(d, S, t, i, sb, 1, x, y, z, rc, ax, ay, az);
        vx = fma(hk, ax, vx); vy = fma(hk, ay, vy); vz = fma(hk, az, vz);
    }
    if (live) { S.vx[t] = vx; S.vy[t] = vy; S.vz[t] = vz; }
    __syncthreads();
    if (!live) return;
    double sx = 0.0, sy = 0.0, sz = 0.0;
    for (int k = 0; k < nm; ++k) {
        const double mk = S.m[sb + k];
        sx = fma(mk, S.vx[sb + k], sx); sy = fma(mk, S.vy[sb + k], sy); sz = fma(mk, S.vz[sb + k], sz);
    }
    const double m0 = d.m0[i / nm], g = 0.5 * h / m0;
    x = fma(g, sx, x); y = fma(g, sy, y); z = fma(g, sz, z);
    d.x0[i] = x; d.y0[i] = y; d.z0[i] = z; d.vx0[i] = vx; d.vy0[i] = vy; d.vz0[i] = vz;
    if (!kepler_drift(d.G * m0, h, x, y, z, vx, vy, vz)) atomicOr(&d.cnt[CI_STATUS], ERRBIT_KEPLER);
    d.x[i] = x; d.y[i] = y; d.z[i] = z; d.vx[i] = vx; d.vy[i] = vy; d.vz[i] = vz;
}
// closing half of the LAST map of a step (no counter reset: the step's encounter data stay readable): Sun kick C(h/2), kick B(hk)
__global__ void __launch_bounds__(128) k_multi_back(DevState d, double h, double hk)
{
    pdl_sync();
    __shared__ MultiSmem S;
    const int nm = d.nm, spb = 128 / nm, t = threadIdx.x;
    const int i = blockIdx.x * spb * nm + t;
    const bool live = t < spb * nm && i < d.ntot;
    double x = 0.0, y = 0.0, z = 0.0, rc = 0.0, vx = 0.0, vy = 0.0, vz = 0.0, m = 0.0;
    if (live) {
        x = d.x[i]; y = d.y[i]; z = d.z[i]; rc = d.rc[i]; vx = d.vx[i]; vy = d.vy[i]; vz = d.vz[i]; m = d.m[i];
        S.m[t] = m; S.vx[t] = vx; S.vy[t] = vy; S.vz[t] = vz; S.rc[t] = rc; S.gm[t] = d.G * m;
    }
    __syncthreads();
    const int sb = (t / nm) * nm;
    if (live) {
        double sx = 0.0, sy = 0.0, sz = 0.0;
        for (int k = 0; k < nm; ++k) {
            const double mk = S.m[sb + k];
            sx = fma(mk, S.vx[sb + k], sx); sy = fma(mk, S.vy[sb + k], sy); sz = fma(mk, S.vz[sb + k], sz);
        }
        const double g = 0.5 * h / d.m0[i / nm];
        x = fma(g, sx, x); y = fma(g, sy, y); z = fma(g, sz, z);
        S.x[t] = x; S.y[t] = y; S.z[t] = z;
    }
    __syncthreads();
    if (!live) return;
    double ax, ay, az;
    multi_pairs(d, S, t, i, sb, 0, x, y, z, rc, ax, ay, az);
    d.x[i] = x; d.y[i] = y; d.z[i] = z;
    d.vx[i] = fma(hk, ax, vx); d.vy[i] = fma(hk, ay, vy); d.vz[i] = fma(hk, az, vz);
}

// =====================================================================================
// Sun kick, operator C (Eq. 3; L196, L232-236, L338, L360-366): s = sum over massive
// bodies of m V (one block per system, fixed-order tree), then q_i += h s / m0 for every
// body of the system, test particles included.
// which: 0 = democratic V as stored; used also for the coordinate maps (with other arrays).
__global__ void k_momentum(DevState d, const double *vx, const double *vy, const double *vz, double fshift)
{
    pdl_sync();
    __shared__ double red[4][32];
    __shared__ double tot[4];
    const int sys = blockIdx.x, base = sys * d.nm * (d.mode == 2 ? 1 : 0);
    double s[4] = {0, 0, 0, 0};
    for (int k = threadIdx.x; k < d.nm; k += blockDim.x) {
        double m = d.m[base + k];
        s[0] = fma(m, vx[base + k], s[0]); s[1] = fma(m, vy[base + k], s[1]); s[2] = fma(m, vz[base + k], s[2]);
        s[3] += m;
    }
#pragma unroll
    for (int c = 0; c < 4; ++c)
        for (int o = 16; o > 0; o >>= 1) s[c] += __shfl_xor_sync(0xffffffffu, s[c], o);
    int w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if ((threadIdx.x & 31) == 0)
        for (int c = 0; c < 4; ++c) red[c][w] = s[c];
    __syncthreads();
    if (threadIdx.x < 4) {
        double t = 0;
        for (int k = 0; k < nw; ++k) t += red[threadIdx.x][k];
        d.psum[4 * sys + threadIdx.x] = t;
        tot[threadIdx.x] = t;
    }
    if (fshift != 0.0) {                                  // the Sun kick of these bodies in the same launch (k_shift's arithmetic)
        __syncthreads();
        const double g = fshift / d.m0[sys];
        for (int k = threadIdx.x; k < d.nm; k += blockDim.x) {
            d.x[base + k] = fma(g, tot[0], d.x[base + k]); d.y[base + k] = fma(g, tot[1], d.y[base + k]);
            d.z[base + k] = fma(g, tot[2], d.z[base + k]);
        }
    }
}
// q += f * psum / m0   (f = h for the Sun kick)
__global__ void k_shift(DevState d, double *ax, double *ay, double *az, double f, int divide_by_total)
{
    pdl_sync();
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= d.ntot) return;
    int sys = system_of(d, i);
    double den = divide_by_total ? d.m0[sys] + d.psum[4 * sys + 3] : d.m0[sys];
    double g = f / den;
    ax[i] = fma(g, d.psum[4 * sys], ax[i]); ay[i] = fma(g, d.psum[4 * sys + 1], ay[i]); az[i] = fma(g, d.psum[4 * sys + 2], az[i]);
}
// root of i in the union-find forest of the group labels (larger roots hang under smaller ones)
__device__ __forceinline__ int uf_find(const int *L, int i)
{
    int p = L[i];
    while (p != i) { i = p; p = L[i]; }
    return i;
}
// link the groups of a and b (atomicMin hooks; safe against concurrent links)
__device__ __forceinline__ void uf_union(int *L, int a, int b)
{
    while (true) {
        a = uf_find(L, a); b = uf_find(L, b);
        if (a == b) break;
        int hi = max(a, b), lo = min(a, b);
        int old = atomicMin(&L[hi], lo);
        if (old == hi) break;
        a = old; b = lo;
    }
}
// Sun kick in one launch (modes 0 and 2): every block forms s = sum m V itself -- mode 0: the block sums the
// massive bodies in a fixed order (at most 8 per thread, then a tree); mode 2: a thread sums the <= 16 bodies of
// its own system -- and shifts its bodies.  reset != 0: thread 0 also zeroes the per-map counters (the map is over).
// hdrift != 0: the Kepler drift over hdrift (operator A, as k_drift) follows in the same thread.
__global__ void __launch_bounds__(256) k_sun(DevState d, double h, int reset, double hdrift)
{
    pdl_sync();
    __shared__ double red[3][8];
    const int i = blockIdx.x * 256 + threadIdx.x;
    if (reset && i == 0) {
        reset_map_counters(d);
    }
    double sx = 0.0, sy = 0.0, sz = 0.0, m0;
    if (d.mode == 2) {
        if (i >= d.ntot) return;
        if (hdrift != 0.0) d.label[i] = i;                    // a new map: every body its own group (k_confirm links them)
        const int sys = i / d.nm, base = sys * d.nm;
        for (int k = 0; k < d.nm; ++k) {
            double m = d.m[base + k];
            sx = fma(m, d.vx[base + k], sx); sy = fma(m, d.vy[base + k], sy); sz = fma(m, d.vz[base + k], sz);
        }
        m0 = d.m0[sys];
    } else {
        // hdrift != 0: the velocities after the kick are in vx0.. (k_kick with to0): this launch only reads them, while
        // vx.. receive the drifted velocities -- a block never sums an array another block of the launch is overwriting
        const double *svx = hdrift != 0.0 ? d.vx0 : d.vx, *svy = hdrift != 0.0 ? d.vy0 : d.vy, *svz = hdrift != 0.0 ? d.vz0 : d.vz;
        double lm[KK_MAXN / 256], lx[KK_MAXN / 256], ly[KK_MAXN / 256], lz[KK_MAXN / 256];
#pragma unroll
        for (int q = 0; q < KK_MAXN / 256; ++q) {                 // all loads in flight together
            const int k = threadIdx.x + 256 * q;
            const bool v = k < d.nm;
            lm[q] = v ? d.m[k] : 0.0; lx[q] = v ? svx[k] : 0.0; ly[q] = v ? svy[k] : 0.0; lz[q] = v ? svz[k] : 0.0;
        }
#pragma unroll
        for (int q = 0; q < KK_MAXN / 256; ++q) { sx = fma(lm[q], lx[q], sx); sy = fma(lm[q], ly[q], sy); sz = fma(lm[q], lz[q], sz); }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            sx += __shfl_xor_sync(0xffffffffu, sx, o); sy += __shfl_xor_sync(0xffffffffu, sy, o); sz += __shfl_xor_sync(0xffffffffu, sz, o);
        }
        if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = sx; red[1][threadIdx.x >> 5] = sy; red[2][threadIdx.x >> 5] = sz; }
        __syncthreads();
        sx = sy = sz = 0.0;
#pragma unroll
        for (int w = 0; w < 8; ++w) { sx += red[0][w]; sy += red[1][w]; sz += red[2][w]; }
        m0 = d.m0[0];
        if (i >= d.ntot) return;
    }
    const double g = h / m0;
    double x = fma(g, sx, d.x[i]), y = fma(g, sy, d.y[i]), z = fma(g, sz, d.z[i]);
    if (hdrift != 0.0) {                                  // opening Sun kick: the Kepler drift follows in the same launch (k_drift)
        double vx, vy, vz;
        if (d.mode == 2) { vx = d.vx[i]; vy = d.vy[i]; vz = d.vz[i]; d.vx0[i] = vx; d.vy0[i] = vy; d.vz0[i] = vz; }
        else { vx = d.vx0[i]; vy = d.vy0[i]; vz = d.vz0[i]; }   // mode 0: already there (read-only in this launch)
        d.x0[i] = x; d.y0[i] = y; d.z0[i] = z;
        if (!kepler_drift(d.G * m0, hdrift, x, y, z, vx, vy, vz)) atomicOr(&d.cnt[CI_STATUS], ERRBIT_KEPLER);
        d.vx[i] = vx; d.vy[i] = vy; d.vz[i] = vz;
    }
    d.x[i] = x; d.y[i] = y; d.z[i] = z;
    if (d.kb && hdrift == 0.0) reinterpret_cast<double4 *>(d.kb)[i] = make_double4(x, y, z, d.G * d.m[i]);   // the j-tile of the kick that follows
}
// Coordinate maps at the ABI in ONE launch (L69): out = in + f * s / den, s = sum m * in over the massive bodies of the
// system, den = m0 (+ sum m if divide_by_total).  Every block forms s itself, in a fixed order: modes 0, 1 as k_sun
// (at most 8 bodies per thread, then a tree), mode 2 a thread sums the bodies of its own system.
__global__ void __launch_bounds__(256) k_coord_map(DevState d, const double *ix, const double *iy, const double *iz,
                                                   double *ox, double *oy, double *oz, double f, int divide_by_total, int init)
{
    pdl_sync();
    __shared__ double red[4][8];
    const int i = blockIdx.x * 256 + threadIdx.x;
    if (init) {                                           // a new state has been loaded (genga_set_state*): every body is what its slot
        if (i == 0) { d.stat[CNT_NEV] = 0; d.stat[CNT_STEPID] = 0; }   // says, no spin, no internal energy, no events, step 0
        if (i < d.nsys) d.U[i] = 0.0;
        if (i < d.ntot) {
            d.kind[i] = (d.mode == 1 && i >= d.nm) ? 1 : 0;
            for (int c = 0; c < 3; ++c) d.spin[(size_t)c * d.np + i] = 0.0;
        }
    }
    double sx = 0.0, sy = 0.0, sz = 0.0, sm = 0.0, m0;
    if (d.mode == 2) {
        if (i >= d.ntot) return;
        const int sys = i / d.nm, base = sys * d.nm;
        for (int k = 0; k < d.nm; ++k) {
            double m = d.m[base + k];
            sx = fma(m, ix[base + k], sx); sy = fma(m, iy[base + k], sy); sz = fma(m, iz[base + k], sz);
            sm += m;
        }
        m0 = d.m0[sys];
    } else {
#pragma unroll
        for (int q = 0; q < KK_MAXN / 256; ++q) {
            const int k = threadIdx.x + 256 * q;
            if (k < d.nm) {
                double m = d.m[k];
                sx = fma(m, ix[k], sx); sy = fma(m, iy[k], sy); sz = fma(m, iz[k], sz);
                sm += m;
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            sx += __shfl_xor_sync(0xffffffffu, sx, o); sy += __shfl_xor_sync(0xffffffffu, sy, o);
            sz += __shfl_xor_sync(0xffffffffu, sz, o); sm += __shfl_xor_sync(0xffffffffu, sm, o);
        }
        if ((threadIdx.x & 31) == 0) {
            red[0][threadIdx.x >> 5] = sx; red[1][threadIdx.x >> 5] = sy; red[2][threadIdx.x >> 5] = sz; red[3][threadIdx.x >> 5] = sm;
        }
        __syncthreads();
        sx = sy = sz = sm = 0.0;
#pragma unroll
        for (int w = 0; w < 8; ++w) { sx += red[0][w]; sy += red[1][w]; sz += red[2][w]; sm += red[3][w]; }
        m0 = d.m0[0];
        if (i >= d.ntot) return;
    }
    const double g = f / (divide_by_total ? m0 + sm : m0);
    ox[i] = fma(g, sx, ix[i]); oy[i] = fma(g, sy, iy[i]); oz[i] = fma(g, sz, iz[i]);
}

// =====================================================================================
// Kepler drift, the analytic part of operator A (Eq. 9; L195, L208-230): one thread per
// body, state kept before the drift for the encounter search and for BS.
__global__ void __launch_bounds__(128) k_drift(DevState d, double h, double hsun)
{
    pdl_sync();
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= d.ntot) return;
    double x = d.x[i], y = d.y[i], z = d.z[i], vx = d.vx[i], vy = d.vy[i], vz = d.vz[i];
    if (hsun != 0.0) {                                    // Sun kick first (k_shift's arithmetic, psum from k_momentum)
        const int sys = system_of(d, i);
        const double g = hsun / d.m0[sys];
        x = fma(g, d.psum[4 * sys], x); y = fma(g, d.psum[4 * sys + 1], y); z = fma(g, d.psum[4 * sys + 2], z);
    }
    d.x0[i] = x; d.y0[i] = y; d.z0[i] = z; d.vx0[i] = vx; d.vy0[i] = vy; d.vz0[i] = vz;
    double mu = d.G * d.m0[system_of(d, i)];
    if (!kepler_drift(mu, h, x, y, z, vx, vy, vz)) atomicOr(&d.cnt[CI_STATUS], ERRBIT_KEPLER);
    d.x[i] = x; d.y[i] = y; d.z[i] = z; d.vx[i] = vx; d.vy[i] = vy; d.vz[i] = vz;
}
// stand-alone drift on caller arrays (genga_kepler_drift)
__global__ void __launch_bounds__(128) k_drift_arrays(long long n, double mu, double h, double *x, double *v, int *status)
{
    pdl_sync();
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double a = x[i], b = x[n + i], c = x[2 * n + i], va = v[i], vb = v[n + i], vc = v[2 * n + i];
    if (!kepler_drift(mu, h, a, b, c, va, vb, vc)) atomicOr(status, ERRBIT_KEPLER);
    x[i] = a; x[n + i] = b; x[2 * n + i] = c; v[i] = va; v[n + i] = vb; v[2 * n + i] = vc;
}

// =====================================================================================
// Encounter search (Eq. 10-12; L200, L276-278): one thread per candidate, confirmed
// pairs appended to the encounter list (warp-aggregated atomic).  Mode 1: a pair with a test
// particle also sets the massive body's bit in the particle's mask and lists the particle once.
__global__ void __launch_bounds__(128) k_confirm(DevState d, double h)
{
    pdl_sync();
    const int nc = min(d.cnt[CI_NCAND], (int)d.cap);
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < nc; e += gridDim.x * blockDim.x) {
        int2 p = d.cand[e];
        int i = p.x, j = p.y;
        double dx = d.x0[j] - d.x0[i], dy = d.y0[j] - d.y0[i], dz = d.z0[j] - d.z0[i];
        double dvx = d.vx0[j] - d.vx0[i], dvy = d.vy0[j] - d.vy0[i], dvz = d.vz0[j] - d.vz0[i];
        double P0 = dx * dx + dy * dy + dz * dz, Pd0 = 2.0 * (dx * dvx + dy * dvy + dz * dvz);
        dx = d.x[j] - d.x[i]; dy = d.y[j] - d.y[i]; dz = d.z[j] - d.z[i];
        dvx = d.vx[j] - d.vx[i]; dvy = d.vy[j] - d.vy[i]; dvz = d.vz[j] - d.vz[i];
        double P1 = dx * dx + dy * dy + dz * dz, Pd1 = 2.0 * (dx * dvx + dy * dvy + dz * dvz);
        double rcij = fmax(d.rc[i], d.rc[j]);
        double D = hermite_min(P0, P1, Pd0, Pd1, h);
        if (D < rcij * rcij) {
            int idx = atomicAdd(&d.cnt[CI_NENC], 1);
            if (idx < d.cap) d.enc[idx] = p;
            else atomicOr(&d.cnt[CI_STATUS], ERRBIT_CAPACITY);
            if (d.mode == 2) uf_union(d.label, i, j);         // multi-system mode: grouping goes with the confirmation
            if (d.mode == 1 && j >= d.nm) {
                unsigned old = atomicOr(&d.tpmask[j - d.nm], 1u << i);
                if (old == 0u) {
                    int k = atomicAdd(&d.cnt[CI_NTP], 1);
                    d.tplist[k] = j;     // at most n_test entries: never overflows
                }
            }
        }
    }
}

// =====================================================================================
// Grouping (L280-284, Appendix): equivalence classes of the encounter graph,
// label = lowest member index.  Union-find with atomicMin hooks (larger root under smaller
// root), then pointer jumping to the root -- the LINK iteration of the Appendix without the
// repeat-until-unchanged sweep.

// exclusive scan of two ints per thread over a 1024-thread block
__device__ __forceinline__ void block_scan2(int v0, int v1, int &e0, int &e1, int &total, int *wsum)
{
    int t = v0 + v1, lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int inc = t;
    for (int o = 1; o < 32; o <<= 1) { int n = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += n; }
    __syncthreads();
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    if (w == 0) {
        int s = wsum[lane], si = s;
        for (int o = 1; o < 32; o <<= 1) { int n = __shfl_up_sync(0xffffffffu, si, o); if (lane >= o) si += n; }
        wsum[lane] = si - s;
        if (lane == 31) wsum[32] = si;
    }
    __syncthreads();
    int base = wsum[w] + inc - t;
    e0 = base; e1 = base + v0; total = wsum[32];
}

// Member lists of the groups of massive bodies (modes 0 and 1; N <= 2048): groups numbered by
// root index, members sorted by body index ("write the members of the groups line by line
// into a matrix", L565 -- here a CSR list), plus `gorder`: the group numbers by DECREASING size
// (counting sort), the order in which the Bulirsch-Stoer kernels take them from their queue so
// that the longest integrations start first.  One block of 1024 threads.
// The labelling itself (the same union-find, in shared memory) runs first in the same block.
__global__ void __launch_bounds__(1024) k_build_groups(DevState d)
{
    pdl_sync();
    __shared__ int lab[2048], sz[2048], E[2048], gst[2048];
    __shared__ __align__(16) int hist[2048];
    __shared__ int wsum[33];
    const int N = d.nm, tid = threadIdx.x, i0 = 2 * tid, i1 = 2 * tid + 1;
    lab[i0] = i0; lab[i1] = i1;
    sz[i0] = 0; sz[i1] = 0; hist[i0] = 0; hist[i1] = 0;
    __syncthreads();
    {
        const int nenc = min(d.cnt[CI_NENC], (int)d.cap);
        for (int e = tid; e < nenc; e += 1024) {
            int2 p = d.enc[e];
            if (d.mode == 1 && p.y >= d.nm) continue;       // particle pairs do not link massive bodies
            int a = p.x, b = p.y;
            while (true) {
                a = uf_find(lab, a); b = uf_find(lab, b);
                if (a == b) break;
                int hi = max(a, b), lo = min(a, b);
                int old = atomicMin(&lab[hi], lo);
                if (old == hi) break;
                a = old; b = lo;
            }
        }
        __syncthreads();
        int r0 = uf_find(lab, i0), r1 = uf_find(lab, i1);   // roots do not change any more: concurrent shortening is safe
        __syncthreads();
        lab[i0] = r0; lab[i1] = r1;
        if (i0 < N) d.label[i0] = r0;
        if (i1 < N) d.label[i1] = r1;
    }
    __syncthreads();
    if (i0 < N) atomicAdd(&sz[lab[i0]], 1);
    if (i1 < N) atomicAdd(&sz[lab[i1]], 1);
    __syncthreads();
    int f0 = i0 < N && sz[lab[i0]] >= 2, f1 = i1 < N && sz[lab[i1]] >= 2;
    int e0, e1, ne, g0, g1, ng, s0, s1, ns;
    block_scan2(f0, f1, e0, e1, ne, wsum);
    if (f0) E[e0] = i0;
    if (f1) E[e1] = i1;
    int r0 = f0 && lab[i0] == i0, r1 = f1 && lab[i1] == i1;
    block_scan2(r0, r1, g0, g1, ng, wsum);
    block_scan2(r0 ? sz[i0] : 0, r1 ? sz[i1] : 0, s0, s1, ns, wsum);
    if (r0) { gst[i0] = s0; d.gstart[g0] = s0; d.gsize[g0] = sz[i0]; atomicAdd(&hist[2048 - sz[i0]], 1); }
    if (r1) { gst[i1] = s1; d.gstart[g1] = s1; d.gsize[g1] = sz[i1]; atomicAdd(&hist[2048 - sz[i1]], 1); }
    __syncthreads();
    // hist[b] = number of groups of 2048 - b bodies -> start of that size class in gorder
    int h0, h1, nh;
    block_scan2(hist[i0], hist[i1], h0, h1, nh, wsum);
    __syncthreads();
    hist[i0] = h0; hist[i1] = h1;
    __syncthreads();
    if (r0) d.gorder[atomicAdd(&hist[2048 - sz[i0]], 1)] = g0;
    if (r1) d.gorder[atomicAdd(&hist[2048 - sz[i1]], 1)] = g1;
    // rank of a member inside its group = members of the same group before it in the (index-ordered) list E;
    // the roots of the listed bodies go to a compact array first (hist is free now) and are scanned 8 at a time
    __syncthreads();
    for (int k = tid; k < ne; k += blockDim.x) hist[k] = lab[E[k]];
    __syncthreads();
    for (int k = tid; k < ne; k += blockDim.x) {
        const int r = hist[k];
        int rank = 0, kk = 0;
        const int4 *h4 = reinterpret_cast<const int4 *>(hist);
        for (; kk + 8 <= k; kk += 8) {
            const int4 a = h4[kk >> 2], b = h4[(kk >> 2) + 1];
            rank += (a.x == r) + (a.y == r) + (a.z == r) + (a.w == r) + (b.x == r) + (b.y == r) + (b.z == r) + (b.w == r);
        }
        for (; kk < k; ++kk) rank += (hist[kk] == r);
        d.gmem[gst[r] + rank] = E[k];
    }
    if (d.mode == 1 && tid < N) {
        unsigned mask = 0u;
        for (int j = 0; j < N; ++j) if (lab[j] == lab[tid]) mask |= 1u << j;
        d.gmask[tid] = mask;
    }
    // groups too large for the cluster layout come first in gorder: their count is the start of
    // the cluster kernels' queues.  The exclusive scan value at the class "S bodies" counts the groups larger than S.
    const int bbig = 2048 - BCB_MAXN, bmid = 2048 - BW_MAXN;
    if (i0 == bbig || i1 == bbig) {
        int nbig = i0 == bbig ? h0 : h1;
        d.cnt[CI_NBIG] = nbig;
        d.cnt[CI_QBIG] = nbig;
    }
    if (i0 == bmid || i1 == bmid) {
        int nmid = i0 == bmid ? h0 : h1;            // groups too large for the warp layout
        d.cnt[CI_NMIDEND] = nmid;
        d.cnt[CI_QSMALL] = nmid;
    }
    if (tid == 0) {
        d.cnt[CI_NGROUPS] = ng;
        d.stat[CNT_GROUPS] += ng;
        d.stat[CNT_CAND] += d.cnt[CI_NCAND];
    }
    int big = (r0 ? sz[i0] : 0) > (r1 ? sz[i1] : 0) ? (r0 ? sz[i0] : 0) : (r1 ? sz[i1] : 0);
    for (int o = 16; o > 0; o >>= 1) big = max(big, __shfl_xor_sync(0xffffffffu, big, o));
    if ((tid & 31) == 0 && big > 0) atomicMax((unsigned long long *)&d.stat[CNT_MAXGROUP], (unsigned long long)big);
}

// =====================================================================================
// Bulirsch-Stoer on the groups of massive bodies (modes 0, 1) of 2..MAXN bodies: one CLUSTER
// of CS CTAs per group, each CTA integrating 8 / CS extrapolation columns (bs_cluster.cuh).  All
// members start from the state before the drift and overwrite the drift result (L163, L301-314).
// Clusters take groups from a queue in order of decreasing size: entries [cnt[qslot], cnt[endslot])
// of gorder (two instantiations run side by side on the two halves of the queue).
template <int MAXN, int THREADS, int LV>
__global__ void __launch_bounds__(THREADS) k_bs_cluster(DevState d, double h, int qslot, int endslot)
{
    pdl_sync();
    extern __shared__ __align__(16) unsigned char bc_raw[];
    using Smem = BcSmem<MAXN, THREADS>;
    Smem &S = *reinterpret_cast<Smem *>(bc_raw);
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank();
    Smem *S0 = cluster.map_shared_rank(&S, 0);
    if (threadIdx.x == 0) {
        S.seq_begin = 0; S.seq_end = 0; S.rec_state = 0;
        for (int k = 0; k < BS_KMAX; ++k) S.ready[k] = 0;
        for (int k = 0; k < 4; ++k) S.lev_result[k] = 0;
    }
    int seq = 0;                                    // round numbers of the cluster's protocol run on from group to group
    const int qend = d.cnt[endslot];
    while (true) {
        if (rank == 0 && threadIdx.x == 0) S.cur = atomicAdd(&d.cnt[qslot], 1);
        cluster.sync();                             // also: everybody has left the previous group, its shared memory may be reused
        const int qi = S0->cur;
        if (qi >= qend) break;
        const int g = d.gorder[qi];
        const int n = d.gsize[g], off = d.gstart[g];
        const BcLane t = bc_lanes<THREADS>(n);
        for (int b = threadIdx.x; b < n; b += THREADS) {
            int i = d.gmem[off + b];
            S.Y[0][b] = d.x0[i]; S.Y[1][b] = d.y0[i]; S.Y[2][b] = d.z0[i];
            S.Y[3][b] = d.vx0[i]; S.Y[4][b] = d.vy0[i]; S.Y[5][b] = d.vz0[i];
            double rc = d.rc[i];
            S.m[b] = d.m[i]; S.rc[b] = rc; S.irc[b] = rc > 0.0 ? 1.0 / (0.9 * rc) : 0.0;
            S.R[b] = d.coll && d.kind[i] != 2 ? d.radius[i] : -1.0;
        }
        int nsteps[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        cluster.sync();                             // S0->cur has been read by everybody (the master may pop the next group)
        const long long t0 = clock64();
        const int ok = bc_integrate<MAXN, THREADS, LV>(S, rank, t, d.G, d.m0[0], h, d.eps, nsteps, seq, d.coll);
        if (ok == 2) {                                  // a collision inside this group: k_bs_generic integrates it again, with the merge
            if (rank == 0 && threadIdx.x == 0) push_redo(d, 0, g, 0);
            continue;
        }
        if (rank == 0) {
            __syncthreads();
            for (int b = threadIdx.x; b < n; b += THREADS) {
                int i = d.gmem[off + b];
                d.x[i] = S.Y[0][b]; d.y[i] = S.Y[1][b]; d.z[i] = S.Y[2][b];
                d.vx[i] = S.Y[3][b]; d.vy[i] = S.Y[4][b]; d.vz[i] = S.Y[5][b];
            }
            if (threadIdx.x == 0) {
                if (!ok) atomicOr(&d.cnt[CI_STATUS], ERRBIT_BS);
                atomicAdd((unsigned long long *)&d.stat[CNT_BSSTEPS], (unsigned long long)nsteps[0]);
                atomicAdd((unsigned long long *)&d.stat[CNT_BSREJECTS], (unsigned long long)nsteps[1]);
                bs_trace(d, n, 1, nsteps, t0, d.gmem[off]);
#ifdef GENGA_BC_PROF
                {   // cycles / 16 by phase: record, rhs, wait, check, publish
                    const int k = atomicAdd(&d.cnt[CI_NTRACE], 2);
                    if (k + 1 < BS_TRACE_CAP) {
                        d.bstrace[k] = make_int4(n | (2 << 16), nsteps[2], nsteps[3], nsteps[4]);
                        d.bstrace[k + 1] = make_int4(n | (3 << 16), nsteps[5], nsteps[6], 0);
                    }
                }
#endif
            }
        }
    }
    cluster.sync();     // nobody leaves while its shared memory may still be read
}
template __global__ void k_bs_cluster<BCB_MAXN, BCB_THREADS, BCB_LV>(DevState, double, int, int);

// Bulirsch-Stoer on the SMALL groups (2..BW_MAXN bodies) of every mode: one block of 4 warps per group, the
// extrapolation columns and several trial step sizes side by side in its lanes (bs_small.cuh).  Blocks take groups
// from a queue:
//   mode 0/1: entries [cnt[CI_QSMALL], cnt[CI_NGROUPS]) of gorder (groups by decreasing size);
//   mode 2  : entries [0, cnt[CI_NGROUPS]) of gorder, each (system, 16-bit member mask);
//   particles (tp = 1, mode 1): entries [0, cnt[CI_NTP]) of tplist; group = {particle} + the massive
//             bodies it meets + their massive groups (L342), only the particle is written back.
__global__ void __launch_bounds__(32 * BW_WARPS) k_bs_warp(DevState d, double h, int tp)
{
    pdl_sync();
    __shared__ BsmSmem W;
    __shared__ int s_qi;
    const int lane = threadIdx.x & 31;
    const int qslot = tp ? CI_QTP : CI_QWARP;
    const int qend = tp ? d.cnt[CI_NTP] : d.cnt[CI_NGROUPS];
    if (!tp && d.mode != 2 && d.cnt[CI_QSMALL] >= qend) return;
    while (true) {
        __syncthreads();                                   // the previous group is finished with s_qi and W
        if (threadIdx.x == 0) s_qi = atomicAdd(&d.cnt[qslot], 1);
        __syncthreads();
        int qi = s_qi;
        if (!tp && d.mode != 2) qi += d.cnt[CI_QSMALL];
        if (qi >= qend) break;
        // ---- members of the group: body index of slot b = lane % 8
        const int b8 = lane & 7;
        int n, i = -1, sys = 0, plabel = 0;
        bool writeback;
        if (tp) {
            const int p = d.tplist[qi];
            unsigned mask = d.tpmask[p - d.nm], fullm = 0u;
            plabel = p;
            for (unsigned mm = mask; mm; mm &= mm - 1) {
                int j = __ffs(mm) - 1;
                fullm |= d.gmask[j];
                plabel = min(plabel, d.label[j]);
            }
            n = __popc(fullm) + 1;
            if (n > BW_MAXN) continue;                     // k_tp_bs<32> takes it
            if (b8 < n - 1) i = __fns(fullm, 0, b8 + 1); else if (b8 == n - 1) i = p;
            writeback = b8 == n - 1;
        } else if (d.mode == 2) {
            sys = d.gorder[2 * qi];
            const unsigned mask = (unsigned)d.gorder[2 * qi + 1];
            n = __popc(mask);
            if (n > BW_MAXN) continue;                     // k_bs_multi takes it
            if (b8 < n) i = sys * d.nm + __fns(mask, 0, b8 + 1);
            writeback = b8 < n;
        } else {
            const int g = d.gorder[qi];
            n = d.gsize[g];
            if (b8 < n) i = d.gmem[d.gstart[g] + b8];
            writeback = b8 < n;
        }
        double Y[6] = {1.0, 0.0, 0.0, 0.0, 1.0, 0.0}, rc = 0.0, m = 0.0;
        if (i >= 0) {
            Y[0] = d.x0[i]; Y[1] = d.y0[i]; Y[2] = d.z0[i]; Y[3] = d.vx0[i]; Y[4] = d.vy0[i]; Y[5] = d.vz0[i];
            rc = d.rc[i]; m = d.m[i];
        }
        if (d.coll && threadIdx.x < 8) {                   // radii for the collision test (a removed body: none)
            W.R[threadIdx.x] = i >= 0 && d.kind[i] != 2 ? d.radius[i] : -1.0;
            W.coll = 1;
        } else if (threadIdx.x == 0) W.coll = 0;
        const double Gm0 = d.G * d.m0[sys];
        int nsteps[2] = {0, 0};
        const long long t0 = clock64();
        int ok;
        if (n <= 4) {
            // segments of 2 or 4 lanes: slot b = lane % S takes body b from lane b of the 8-slot layout
            const int src = n == 2 ? (lane & 1) : (lane & 3);
#pragma unroll
            for (int c = 0; c < 6; ++c) Y[c] = __shfl_sync(0xffffffffu, Y[c], src);
            rc = __shfl_sync(0xffffffffu, rc, src); m = __shfl_sync(0xffffffffu, m, src);
            if (n == 2) ok = bsm_integrate<2, BW_WARPS>(W, n, Gm0, rc, m, d.G, Y, h, d.eps, nsteps);
            else ok = bsm_integrate<4, BW_WARPS>(W, n, Gm0, rc, m, d.G, Y, h, d.eps, nsteps);
        } else {
            ok = bsm_integrate<8, BW_WARPS>(W, n, Gm0, rc, m, d.G, Y, h, d.eps, nsteps);
        }
        if (ok == 2) {                                     // a collision inside this group: k_bs_generic integrates it again, with the merge
            if (threadIdx.x == 0) {
                if (tp) push_redo(d, 1, d.tplist[qi], 0);
                else if (d.mode == 2) push_redo(d, 2, sys, d.gorder[2 * qi + 1]);
                else push_redo(d, 0, d.gorder[qi], 0);
            }
            continue;
        }
        if (threadIdx.x < 8 && writeback) {
            d.x[i] = Y[0]; d.y[i] = Y[1]; d.z[i] = Y[2]; d.vx[i] = Y[3]; d.vy[i] = Y[4]; d.vz[i] = Y[5];
            if (tp) d.label[i] = plabel;
        }
        if (threadIdx.x == 0) {
            if (!ok) atomicOr(&d.cnt[CI_STATUS], ERRBIT_BS);
            atomicAdd((unsigned long long *)&d.stat[CNT_BSSTEPS], (unsigned long long)nsteps[0]);
            atomicAdd((unsigned long long *)&d.stat[CNT_BSREJECTS], (unsigned long long)nsteps[1]);
            if (tp || d.mode == 2) {
                atomicAdd((unsigned long long *)&d.stat[CNT_GROUPS], 1ull);
                atomicMax((unsigned long long *)&d.stat[CNT_MAXGROUP], (unsigned long long)n);
            }
            bs_trace(d, n, 0, nsteps, t0, i);
        }
    }
}

// Multi-system mode: the groups of every system as one queue for k_bs_warp.  One thread per body; a
// root (label = own index) with at least one other member appends (system, member mask).
__global__ void k_list_groups_multi(DevState d)
{
    pdl_sync();
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (d.cnt[CI_NENC] == 0 || i >= d.ntot) return;
    const int root = uf_find(d.label, i);                     // flatten on the way (values only move towards the root)
    d.label[i] = root;
    if (root != i) return;
    const int nm = d.nm, sys = i / nm, base = sys * nm;
    unsigned mask = 0u;
    for (int k = 0; k < nm; ++k) if (uf_find(d.label, base + k) == i) mask |= 1u << k;
    if (__popc(mask) < 2) return;
    int slot = atomicAdd(&d.cnt[CI_NGROUPS], 1);
    d.gorder[2 * slot] = sys; d.gorder[2 * slot + 1] = (int)mask;
    if (__popc(mask) > BW_MAXN) atomicAdd(&d.cnt[CI_NBIG], 1);
}

// Groups larger than a warp: one block per group, tableau in global scratch.
__global__ void __launch_bounds__(256) k_bs_block(DevState d, double h)
{
    pdl_sync();
    __shared__ double red[32];
    __shared__ int nsteps[2];
    if (d.cnt[CI_NBIG] == 0) return;
    const int ng = d.cnt[CI_NGROUPS];
    for (int g = blockIdx.x; g < ng; g += gridDim.x) {
        const int nb = d.gsize[g];
        if (nb <= BCB_MAXN) continue;
        if (d.coll) { if (threadIdx.x == 0) push_redo(d, 0, g, 0); continue; }   // collisions: the generic layout takes it
        const int off = d.gstart[g];
        if (threadIdx.x == 0) { nsteps[0] = 0; nsteps[1] = 0; }
        for (int b = threadIdx.x; b < nb; b += blockDim.x) {
            int i = d.gmem[off + b];
            d.bss.arr(BSA_Y + 0)[off + b] = d.x0[i]; d.bss.arr(BSA_Y + 1)[off + b] = d.y0[i]; d.bss.arr(BSA_Y + 2)[off + b] = d.z0[i];
            d.bss.arr(BSA_Y + 3)[off + b] = d.vx0[i]; d.bss.arr(BSA_Y + 4)[off + b] = d.vy0[i]; d.bss.arr(BSA_Y + 5)[off + b] = d.vz0[i];
            d.bss.arr(BSA_M)[off + b] = d.m[i]; d.bss.arr(BSA_RC)[off + b] = d.rc[i];
        }
        bool ok = bs_block(d.bss, off, nb, d.G, d.m0[0], h, d.eps, red, nsteps);
        __syncthreads();
        for (int b = threadIdx.x; b < nb; b += blockDim.x) {
            int i = d.gmem[off + b];
            d.x[i] = d.bss.arr(BSA_Y + 0)[off + b]; d.y[i] = d.bss.arr(BSA_Y + 1)[off + b]; d.z[i] = d.bss.arr(BSA_Y + 2)[off + b];
            d.vx[i] = d.bss.arr(BSA_Y + 3)[off + b]; d.vy[i] = d.bss.arr(BSA_Y + 4)[off + b]; d.vz[i] = d.bss.arr(BSA_Y + 5)[off + b];
        }
        if (threadIdx.x == 0) {
            if (!ok) atomicOr(&d.cnt[CI_STATUS], ERRBIT_BS);
            atomicAdd((unsigned long long *)&d.stat[CNT_BSSTEPS], (unsigned long long)nsteps[0]);
                atomicAdd((unsigned long long *)&d.stat[CNT_BSREJECTS], (unsigned long long)nsteps[1]);
        }
        __syncthreads();
    }
}

// Test-particle groups (L342): {particle} + the massive bodies it meets + their massive
// groups; everything integrated from the state before the drift, only the particle is
// written back.  One team of TW lanes per listed particle; teams whose group does not fit
// TW (or fits the next smaller instantiation, `lo`) skip.
template <int TW>
__global__ void __launch_bounds__(128) k_tp_bs(DevState d, double h, int lo)
{
    pdl_sync();
    constexpr int TPB = 128 / TW;                       // teams per block
    __shared__ TeamSmem<TW> sm[TPB];
    const int ntp = d.cnt[CI_NTP];
    const int team = threadIdx.x / TW, lane = threadIdx.x % TW;
    const int lane32 = threadIdx.x & 31;
    const unsigned tmask = TW == 32 ? 0xffffffffu : (((1u << TW) - 1u) << (lane32 - lane));
    WarpTeam<TW> t{tmask, lane};
    for (int k = blockIdx.x * TPB + team; k < ntp; k += gridDim.x * TPB) {
        const int p = d.tplist[k];
        unsigned mask = d.tpmask[p - d.nm], full = 0u;
        int lab = p;
        for (unsigned mm = mask; mm; mm &= mm - 1) {
            int j = __ffs(mm) - 1;
            full |= d.gmask[j];
            lab = min(lab, d.label[j]);
        }
        const int nb = __popc(full) + 1;
        if (nb > TW || nb <= lo) continue;            // 32 massive bodies + the particle: k_tp_bs_big
        if (d.coll) { if (lane == 0) push_redo(d, 1, p, 0); continue; }      // collisions: the generic layout takes it
        const bool active = lane < nb;
        int i = p;
        if (lane < nb - 1) {                         // lane-th set bit of full
            unsigned mm = full;
            for (int c = 0; c < lane; ++c) mm &= mm - 1;
            i = __ffs(mm) - 1;
        }
        double q[3] = {1.0, 0.0, 0.0}, V[3] = {0.0, 1.0, 0.0}, rc = 0.0;
        t.sync();
        sm[team].m[lane] = 0.0; sm[team].rc[lane] = 0.0; sm[team].irc[lane] = 0.0;
        if (active) {
            q[0] = d.x0[i]; q[1] = d.y0[i]; q[2] = d.z0[i]; V[0] = d.vx0[i]; V[1] = d.vy0[i]; V[2] = d.vz0[i];
            rc = d.rc[i];
            sm[team].m[lane] = d.m[i]; sm[team].rc[lane] = rc; sm[team].irc[lane] = rc > 0.0 ? 1.0 / (0.9 * rc) : 0.0;
        }
        t.sync();
        int nsteps[2] = {0, 0};
        unsigned srcmask = nb >= 32 ? 0xffffffffu : ((1u << nb) - 1u);
        bool ok = bs_team<TW>(t, sm[team], nb, active, srcmask, d.G, d.m0[0], rc, q, V, h, d.eps, nsteps);
        if (lane == nb - 1) {
            d.x[p] = q[0]; d.y[p] = q[1]; d.z[p] = q[2]; d.vx[p] = V[0]; d.vy[p] = V[1]; d.vz[p] = V[2];
            d.label[p] = lab;
            if (!ok) atomicOr(&d.cnt[CI_STATUS], ERRBIT_BS);
            atomicAdd((unsigned long long *)&d.stat[CNT_BSSTEPS], (unsigned long long)nsteps[0]);
                atomicAdd((unsigned long long *)&d.stat[CNT_BSREJECTS], (unsigned long long)nsteps[1]);
            atomicAdd((unsigned long long *)&d.stat[CNT_GROUPS], 1ull);
            atomicMax((unsigned long long *)&d.stat[CNT_MAXGROUP], (unsigned long long)nb);
        }
    }
}
template __global__ void k_tp_bs<32>(DevState, double, int);

// Test-particle groups of 33 bodies: all 32 massive bodies of the mode's maximum (L188) in one group, plus the particle
// (L342).  One more body than a warp holds: one block per listed particle with the tableau in global scratch (bs_block,
// 64 entries per block); rare, so the slow layout is enough.  Only the particle is written back.
__global__ void __launch_bounds__(64) k_tp_bs_big(DevState d, double h)
{
    pdl_sync();
    __shared__ double red[32];
    __shared__ int nsteps[2];
    const int ntp = d.cnt[CI_NTP];
    const int off = blockIdx.x * 64;
    for (int k = blockIdx.x; k < ntp; k += gridDim.x) {
        const int p = d.tplist[k];
        unsigned mask = d.tpmask[p - d.nm], full = 0u;
        int lab = p;
        for (unsigned mm = mask; mm; mm &= mm - 1) {
            int j = __ffs(mm) - 1;
            full |= d.gmask[j];
            lab = min(lab, d.label[j]);
        }
        const int nb = __popc(full) + 1;
        if (nb <= 32) continue;                           // k_bs_warp / k_tp_bs<32> (uniform over the block)
        if (d.coll) { if (threadIdx.x == 0) push_redo(d, 1, p, 0); continue; }
        if (threadIdx.x == 0) { nsteps[0] = 0; nsteps[1] = 0; }
        for (int b = threadIdx.x; b < nb; b += blockDim.x) {
            const int i = b < nb - 1 ? __fns(full, 0, b + 1) : p;
            d.bss.arr(BSA_Y + 0)[off + b] = d.x0[i]; d.bss.arr(BSA_Y + 1)[off + b] = d.y0[i]; d.bss.arr(BSA_Y + 2)[off + b] = d.z0[i];
            d.bss.arr(BSA_Y + 3)[off + b] = d.vx0[i]; d.bss.arr(BSA_Y + 4)[off + b] = d.vy0[i]; d.bss.arr(BSA_Y + 5)[off + b] = d.vz0[i];
            d.bss.arr(BSA_M)[off + b] = d.m[i]; d.bss.arr(BSA_RC)[off + b] = d.rc[i];
        }
        const bool ok = bs_block(d.bss, off, nb, d.G, d.m0[0], h, d.eps, red, nsteps);
        __syncthreads();
        if (threadIdx.x == 0) {
            const int b = nb - 1;
            d.x[p] = d.bss.arr(BSA_Y + 0)[off + b]; d.y[p] = d.bss.arr(BSA_Y + 1)[off + b]; d.z[p] = d.bss.arr(BSA_Y + 2)[off + b];
            d.vx[p] = d.bss.arr(BSA_Y + 3)[off + b]; d.vy[p] = d.bss.arr(BSA_Y + 4)[off + b]; d.vz[p] = d.bss.arr(BSA_Y + 5)[off + b];
            d.label[p] = lab;
            if (!ok) atomicOr(&d.cnt[CI_STATUS], ERRBIT_BS);
            atomicAdd((unsigned long long *)&d.stat[CNT_BSSTEPS], (unsigned long long)nsteps[0]);
                atomicAdd((unsigned long long *)&d.stat[CNT_BSREJECTS], (unsigned long long)nsteps[1]);
            atomicAdd((unsigned long long *)&d.stat[CNT_GROUPS], 1ull);
            atomicMax((unsigned long long *)&d.stat[CNT_MAXGROUP], (unsigned long long)nb);
        }
        __syncthreads();
    }
}

// Bulirsch-Stoer WITH collisions (L316-328): one block per listed group, any size, tableau in global scratch (bs_block).
// The fast layouts only notice that a pair of a group collides in an accepted step (same test, same steps) and hand the
// group over; here it is integrated again from the state before the drift, and the pair merges at the end of that
// step.  pass 0: particle groups (only the particle is written back; the massive bodies' merges are re-enacted silently,
// L342) and multi-system groups; pass 1: groups of massive bodies of modes 0, 1, which change masses the particle groups
// must still see unchanged.
__global__ void __launch_bounds__(256) k_bs_generic(DevState d, double h, int pass)
{
    pdl_sync();
    __shared__ double red[32];
    __shared__ int nsteps[2];
    const int nredo = min(d.cnt[CI_NREDO], (int)d.cap);
    for (int e = blockIdx.x; e < nredo; e += gridDim.x) {
        const int2 en = d.redo[e];
        const int kind = (unsigned)en.x >> 28, id = en.x & 0x0fffffff;
        if ((kind == 0) != (pass == 1)) continue;
        int nb, off, sys = 0, p = -1, lab = 0;
        unsigned full = 0u;
        const BsScratch &S = kind == 0 ? d.genA : d.genB;
        if (kind == 0) { nb = d.gsize[id]; off = d.gstart[id]; }
        else if (kind == 1) {
            p = id; lab = p;
            for (unsigned mm = d.tpmask[p - d.nm]; mm; mm &= mm - 1) {
                const int j = __ffs(mm) - 1;
                full |= d.gmask[j];
                lab = min(lab, d.label[j]);
            }
            nb = __popc(full) + 1; off = blockIdx.x * 64;
        } else { sys = id; full = (unsigned)en.y; nb = __popc(full); off = blockIdx.x * 64; }
        const int base = d.mode == 2 ? sys * d.nm : 0;
        if (threadIdx.x == 0) { nsteps[0] = 0; nsteps[1] = 0; }
        for (int b = threadIdx.x; b < nb; b += blockDim.x) {
            const int i = kind == 0 ? d.gmem[off + b] : kind == 1 ? (b < nb - 1 ? __fns(full, 0, b + 1) : p) : base + __fns(full, 0, b + 1);
            S.arr(BSA_Y + 0)[off + b] = d.x0[i]; S.arr(BSA_Y + 1)[off + b] = d.y0[i]; S.arr(BSA_Y + 2)[off + b] = d.z0[i];
            S.arr(BSA_Y + 3)[off + b] = d.vx0[i]; S.arr(BSA_Y + 4)[off + b] = d.vy0[i]; S.arr(BSA_Y + 5)[off + b] = d.vz0[i];
            S.arr(BSA_M)[off + b] = d.m[i]; S.arr(BSA_RC)[off + b] = d.rc[i];
            S.arr(BSA_R)[off + b] = d.radius[i]; S.arr(BSA_KIND)[off + b] = (double)d.kind[i];
            for (int c = 0; c < 3; ++c) S.arr(BSA_SPIN + c)[off + b] = d.spin[(size_t)c * d.np + i];
            S.arr(BSA_GIDX)[off + b] = (double)(i - base);
        }
        BsColl cc;
        cc.ev = d.ev; cc.evcap = d.evcap; cc.nev = (unsigned long long *)&d.stat[CNT_NEV]; cc.U = d.U + sys;
        cc.step_id = (double)d.stat[CNT_STEPID]; cc.base = base; cc.record_massive = kind != 1;
        const bool ok = bs_block(S, off, nb, d.G, d.m0[sys], h, d.eps, red, nsteps, &cc);
        __syncthreads();
        for (int b = threadIdx.x; b < nb; b += blockDim.x) {
            const int i = kind == 0 ? d.gmem[off + b] : kind == 1 ? (b < nb - 1 ? __fns(full, 0, b + 1) : p) : base + __fns(full, 0, b + 1);
            if (kind == 1 && b < nb - 1) continue;                   // only the particle (L342)
            d.x[i] = S.arr(BSA_Y + 0)[off + b]; d.y[i] = S.arr(BSA_Y + 1)[off + b]; d.z[i] = S.arr(BSA_Y + 2)[off + b];
            d.vx[i] = S.arr(BSA_Y + 3)[off + b]; d.vy[i] = S.arr(BSA_Y + 4)[off + b]; d.vz[i] = S.arr(BSA_Y + 5)[off + b];
            d.m[i] = S.arr(BSA_M)[off + b]; d.radius[i] = S.arr(BSA_R)[off + b]; d.kind[i] = (int)S.arr(BSA_KIND)[off + b];
            for (int c = 0; c < 3; ++c) d.spin[(size_t)c * d.np + i] = S.arr(BSA_SPIN + c)[off + b];
            if (kind == 1) d.label[i] = lab;
        }
        if (threadIdx.x == 0) {
            if (!ok) atomicOr(&d.cnt[CI_STATUS], ERRBIT_BS);
            atomicAdd((unsigned long long *)&d.stat[CNT_BSSTEPS], (unsigned long long)nsteps[0]);
            atomicAdd((unsigned long long *)&d.stat[CNT_BSREJECTS], (unsigned long long)nsteps[1]);
            if (kind != 0) {
                atomicAdd((unsigned long long *)&d.stat[CNT_GROUPS], 1ull);
                atomicMax((unsigned long long *)&d.stat[CNT_MAXGROUP], (unsigned long long)nb);
            }
        }
        __syncthreads();
    }
}

// End of a time step with collisions / ejections switched on: ejections (L330-332: a body farther from the central mass
// than Rcut or closer than RcutSun is reported and removed), the stop of a system with fewer than Nmin bodies left
// (L378-384: all its bodies are removed), the step counter of the event records.  One thread per system does the
// system's bodies in index order (events of a system in a fixed order); removed bodies are parked like the ghosts.
__device__ inline void remove_body(const DevState &d, int i, int base, int sys, int kev)
{
    const unsigned long long slot = atomicAdd((unsigned long long *)&d.stat[CNT_NEV], 1ull);
    if ((long long)slot < d.evcap) {
        double *e = d.ev + GENGA_EV * slot;
        for (int k = 0; k < GENGA_EV; ++k) e[k] = 0.0;
        e[0] = (double)d.stat[CNT_STEPID]; e[1] = kev; e[2] = i; e[3] = -1.0; e[4] = d.m[i]; e[6] = d.radius[i];
        e[8] = d.x[i]; e[9] = d.y[i]; e[10] = d.z[i]; e[11] = d.vx[i]; e[12] = d.vy[i]; e[13] = d.vz[i];
        for (int c = 0; c < 3; ++c) e[21 + c] = d.spin[(size_t)c * d.np + i];
    }
    const double Rp = 1000.0 * (double)(i - base + 1);
    d.m[i] = 0.0; d.radius[i] = 0.0; d.kind[i] = 2;
    for (int c = 0; c < 3; ++c) d.spin[(size_t)c * d.np + i] = 0.0;
    d.x[i] = Rp; d.y[i] = 0.0; d.z[i] = 0.0;
    d.vx[i] = 0.0; d.vy[i] = sqrt(d.G * d.m0[sys] / Rp); d.vz[i] = 0.0;
    if (d.kb && i < d.nm) reinterpret_cast<double4 *>(d.kb)[i] = make_double4(Rp, 0.0, 0.0, 0.0);
    d.cnt[CI_S2PMISS] = 1;                                        // positions changed after the closing kick: its stored sums are void
}
__global__ void k_end_step(DevState d)
{
    pdl_sync();
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (d.mode == 2) {
        if (t < d.nsys) {
            const int base = t * d.nm;
            int left = 0;
            for (int k = 0; k < d.nm; ++k) {
                const int i = base + k;
                if (d.kind[i] == 2) continue;
                const double r2 = d.x[i] * d.x[i] + d.y[i] * d.y[i] + d.z[i] * d.z[i];
                if (d.rcut2 > 0.0 && r2 > d.rcut2) remove_body(d, i, base, t, 2);
                else if (d.rcutsun2 > 0.0 && r2 < d.rcutsun2) remove_body(d, i, base, t, 3);
                else ++left;
            }
            if (d.nmin > 0 && left < d.nmin && left > 0)
                for (int k = 0; k < d.nm; ++k) if (d.kind[base + k] != 2) remove_body(d, base + k, base, t, 4);
        }
    } else {
        // massive bodies and particles: one thread per body; the stop of the (single) system by thread 0 of a second launch
        if (t < d.ntot && d.kind[t] != 2) {
            const double r2 = d.x[t] * d.x[t] + d.y[t] * d.y[t] + d.z[t] * d.z[t];
            if (d.rcut2 > 0.0 && r2 > d.rcut2) remove_body(d, t, 0, 0, 2);
            else if (d.rcutsun2 > 0.0 && r2 < d.rcutsun2) remove_body(d, t, 0, 0, 3);
        }
    }
}
// single system (modes 0, 1): the stop at fewer than Nmin massive bodies, and the step counter
__global__ void k_end_step2(DevState d)
{
    pdl_sync();
    if (d.mode != 2 && d.nmin > 0) {
        __shared__ int left;
        if (threadIdx.x == 0) left = 0;
        __syncthreads();
        int mine = 0;
        for (int i = threadIdx.x; i < d.nm; i += blockDim.x) mine += d.kind[i] != 2;
        atomicAdd(&left, mine);
        __syncthreads();
        if (left < d.nmin && left > 0 && threadIdx.x == 0)
            for (int i = 0; i < d.ntot; ++i) if (d.kind[i] != 2) remove_body(d, i, 0, 0, 4);
    }
    if (threadIdx.x == 0) d.stat[CNT_STEPID] += 1;
}

// Multi-system mode (L372-376), groups of more than BW_MAXN bodies (the others: k_bs_warp): 16 lanes
// per system; the groups of a system are the sets of equal labels among its bodies.
__global__ void __launch_bounds__(128) k_bs_multi(DevState d, double h)
{
    pdl_sync();
    constexpr int TW = 16, TPB = 128 / TW;
    __shared__ TeamSmem<TW> sm[TPB];
    if (d.cnt[CI_NBIG] == 0) return;
    const int team = threadIdx.x / TW, lane = threadIdx.x % TW, lane32 = threadIdx.x & 31;
    const unsigned tmask = 0xffffu << (lane32 - lane);
    WarpTeam<TW> t{tmask, lane};
    const int sys = blockIdx.x * TPB + team;
    if (sys >= d.nsys) return;
    const int nm = d.nm, base = sys * nm;
    const bool have = lane < nm;
    const int i = base + lane;
    int lab = have ? d.label[i] - base : -1 - lane;
    // lanes of my group
    unsigned grp = 0u;
    for (int j = 0; j < TW; ++j) {
        int lj = __shfl_sync(tmask, lab, j, TW);
        if (lj == lab) grp |= 1u << j;
    }
    unsigned todo = __ballot_sync(tmask, have && __popc(grp) > BW_MAXN && lab == lane) >> (lane32 - lane) & 0xffffu;  // roots of groups too large for k_bs_warp
    if (todo == 0u) return;
    double rc = have ? d.rc[i] : 0.0;
    sm[team].m[lane] = have ? d.m[i] : 0.0; sm[team].rc[lane] = rc; sm[team].irc[lane] = rc > 0.0 ? 1.0 / (0.9 * rc) : 0.0;
    t.sync();
    int ngroups = 0, nsteps_tot = 0, nrej_tot = 0, big = 0;
    bool ok = true;
    while (todo) {
        int root = __ffs(todo) - 1;
        todo &= todo - 1;
        unsigned gm = __shfl_sync(tmask, grp, root, TW);
        if (d.coll) { if (lane == 0) push_redo(d, 2, sys, (int)gm); continue; }   // collisions: the generic layout takes it
        bool active = (gm >> lane) & 1u;
        double q[3] = {1.0, 0.0, 0.0}, V[3] = {0.0, 1.0, 0.0};
        if (active) { q[0] = d.x0[i]; q[1] = d.y0[i]; q[2] = d.z0[i]; V[0] = d.vx0[i]; V[1] = d.vy0[i]; V[2] = d.vz0[i]; }
        int nsteps[2] = {0, 0};
        ok = bs_team<TW>(t, sm[team], TW, active, gm, d.G, d.m0[sys], rc, q, V, h, d.eps, nsteps) && ok;
        if (active) { d.x[i] = q[0]; d.y[i] = q[1]; d.z[i] = q[2]; d.vx[i] = V[0]; d.vy[i] = V[1]; d.vz[i] = V[2]; }
        ++ngroups; nsteps_tot += nsteps[0]; nrej_tot += nsteps[1]; big = max(big, __popc(gm));
    }
    if (lane == 0) {
        if (!ok) atomicOr(&d.cnt[CI_STATUS], ERRBIT_BS);
        atomicAdd((unsigned long long *)&d.stat[CNT_BSSTEPS], (unsigned long long)nsteps_tot);
        atomicAdd((unsigned long long *)&d.stat[CNT_BSREJECTS], (unsigned long long)nrej_tot);
        atomicAdd((unsigned long long *)&d.stat[CNT_GROUPS], (unsigned long long)ngroups);
        atomicMax((unsigned long long *)&d.stat[CNT_MAXGROUP], (unsigned long long)big);
    }
}

// =====================================================================================
// Energy and angular momentum (Eq. 1-3 summed, L73-80; L225): one block per system.
// out[sys][0] = E, out[sys][1..3] = L.
__global__ void __launch_bounds__(1024) k_energy(DevState d, double *out)
{
    pdl_sync();
    __shared__ double red[8][32];
    const int sys = blockIdx.x, nm = d.nm, base = d.mode == 2 ? sys * nm : 0;
    const double m0 = d.m0[sys];
    double s[8] = {0, 0, 0, 0, 0, 0, 0, 0};   // kin, pot0, pair, px, py, pz | Lx.. in second pass
    double lx = 0, ly = 0, lz = 0;
    for (int k = threadIdx.x; k < nm; k += blockDim.x) {
        int i = base + k;
        double m = d.m[i], x = d.x[i], y = d.y[i], z = d.z[i], vx = d.vx[i], vy = d.vy[i], vz = d.vz[i];
        s[0] += 0.5 * m * (vx * vx + vy * vy + vz * vz);
        s[1] -= d.G * m0 * m / sqrt(x * x + y * y + z * z);
        s[3] += m * vx; s[4] += m * vy; s[5] += m * vz;
        lx += m * (y * vz - z * vy); ly += m * (z * vx - x * vz); lz += m * (x * vy - y * vx);
        double pp = 0.0;
        for (int kk = k + 1; kk < nm; ++kk) {
            int j = base + kk;
            double dx = d.x[j] - x, dy = d.y[j] - y, dz = d.z[j] - z;
            pp += d.m[j] / sqrt(dx * dx + dy * dy + dz * dz);
        }
        s[2] -= d.G * m * pp;
    }
    s[6] = lx; s[7] = ly;
    double extra = lz;
    for (int c = 0; c < 8; ++c)
        for (int o = 16; o > 0; o >>= 1) s[c] += __shfl_xor_sync(0xffffffffu, s[c], o);
    for (int o = 16; o > 0; o >>= 1) extra += __shfl_xor_sync(0xffffffffu, extra, o);
    __shared__ double red2[32];
    int w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if ((threadIdx.x & 31) == 0) { for (int c = 0; c < 8; ++c) red[c][w] = s[c]; red2[w] = extra; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double t[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
        for (int k = 0; k < nw; ++k) { for (int c = 0; c < 8; ++c) t[c] += red[c][k]; t[8] += red2[k]; }
        out[4 * sys] = t[0] + (t[3] * t[3] + t[4] * t[4] + t[5] * t[5]) / (2.0 * m0) + t[1] + t[2];
        out[4 * sys + 1] = t[6]; out[4 * sys + 2] = t[7]; out[4 * sys + 3] = t[8];
    }
}

// FP64 peak probe: 8 independent DFMA chains per thread, 2 flop per DFMA.  Used only by
// genga_fp64_probe to measure the denominator of the ALU roofline on the device at hand.
__global__ void __launch_bounds__(256) k_fp64_probe(double *out, int iters)
{
    pdl_sync();
    double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double b = 1.0000001, c = 1e-9;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            a0 = fma(a0, b, c); a1 = fma(a1, b, c); a2 = fma(a2, b, c); a3 = fma(a3, b, c);
            a4 = fma(a4, b, c); a5 = fma(a5, b, c); a6 = fma(a6, b, c); a7 = fma(a7, b, c);
        }
    }
    double r = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (r == 0.12345) out[threadIdx.x] = r;      // never true: keeps the chains alive without a per-thread output array
}

// The reciprocal routines of common.cuh on caller arrays (genga_eval_fast): the bias test of tests/test_gpu_fastmath.py.
__global__ void k_eval_fast(int which, long long n, const double *in, double *out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double x = in[i];
    out[i] = which == 0 ? rsqrt_fast(x) : which == 1 ? rinv3_fast(x) : rcp_fast(x);
}

// labels for genga_encounters: body's own index unless it is in a group
__global__ void k_export_labels(DevState d, int *out)
{
    pdl_sync();
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= d.ntot) return;
    int l = i;
    if (d.mode != 1 || i < d.nm) l = d.label[i];
    else if (d.tpmask[i - d.nm] != 0u) l = d.label[i];
    out[i] = l;
}

}  // namespace genga
