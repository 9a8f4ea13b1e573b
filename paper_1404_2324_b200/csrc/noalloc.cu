// genga_kick_accel_noalloc: the kick accelerations of operator B (Eq. 2 L76 with the changeover weight W = K - r dK/dr,
// Eq. 4-8) for callers that cannot allocate -- code under CUDA graph capture, tight serving loops, harnesses that
// forbid cudaMalloc.  It is a variant of k_kick (kernels.cu) whose scratch memory (the packed body records that k_rcrit
// writes into the workspace for k_kick, and the partial sums of the j slices) lives in ONE file-scope device array
// instead of a caller-provided workspace.  The entry point calls no cudaMalloc, cudaFree or allocating library routine.
//
// The array: GENGA_NOALLOC_SCRATCH_BYTES (848 KiB) per GPU that loads the library, held until the process exits.
// Every call on a device shares it, and it keeps the last call's contents.  Nothing in it has to start at zero: every
// word a call reads (records 0..n-1, partial sums [slice][component][0..n-1]) is written earlier by the same call, no
// atomics, no counters; so nothing is cleared.  Two calls that overlap on the GPU (different streams, or concurrent
// graph launches) RACE on it: callers serialise them.
//
// In host code the name g_na_scratch is a host-side stand-in, not a device address; the address the kernels get comes
// from cudaGetSymbolAddress, looked up once per device with that device current (na_scratch_ptr).
#include <cuda_runtime.h>
#include <mutex>
#include <stdint.h>
#include <stdio.h>

#include "../../include/genga.h"
#include "common.cuh"

namespace genga {

constexpr int NA_MAXN = GENGA_NOALLOC_MAX_BODIES;       // 2048: the largest system of the massive mode
constexpr int NA_SLICES = 16;                            // the j loop is cut into 16 slices: blocks (i tile, j slice)
constexpr int NA_THREADS = 128;

struct __align__(32) NaBody { double x, y, z, gm; };

struct NaScratch {
    NaBody body[NA_MAXN];                                // 64 KiB: x, y, z, G m_j
    double rc[NA_MAXN];                                  // 16 KiB: critical radii
    double part[NA_SLICES][3][NA_MAXN];                  // 768 KiB: partial sums of slice s, written before they are read
};
static_assert(sizeof(NaScratch) == GENGA_NOALLOC_SCRATCH_BYTES, "the header states the size of the scratch array");

static __device__ __align__(256) unsigned char g_na_scratch[sizeof(NaScratch)];

// ---- stage 1: pack the caller's arrays into the scratch records (what k_rcrit does for k_kick)
__global__ void __launch_bounds__(NA_THREADS) k_na_pack(NaScratch *S, int n, double G, const double *m, const double *x, const double *rc)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    NaBody b;
    b.x = x[i]; b.y = x[n + i]; b.z = x[2 * n + i]; b.gm = G * m[i];
    S->body[i] = b;
    S->rc[i] = rc[i];
}

// ---- stage 2: block (i tile, j slice): a_i restricted to the bodies j of the slice, in index order
__global__ void __launch_bounds__(NA_THREADS) k_na_pairs(NaScratch *S, int n)
{
    __shared__ NaBody sb[NA_MAXN / NA_SLICES];
    __shared__ double src[NA_MAXN / NA_SLICES];
    const int per = (n + NA_SLICES - 1) / NA_SLICES;     // bodies per slice (<= 128)
    const int s = blockIdx.y, j0 = s * per, j1 = min(n, j0 + per);
    for (int k = threadIdx.x; k < j1 - j0; k += blockDim.x) { sb[k] = S->body[j0 + k]; src[k] = S->rc[j0 + k]; }
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const NaBody me = S->body[i];
    const double my_rc = S->rc[i];
    double ax = 0.0, ay = 0.0, az = 0.0;
    for (int k = 0; k < j1 - j0; ++k) {
        if (j0 + k == i) continue;
        const NaBody o = sb[k];
        const double dx = o.x - me.x, dy = o.y - me.y, dz = o.z - me.z;
        const double r2 = dx * dx + dy * dy + dz * dz;
        const double r = sqrt(r2);
        const double w = kick_weight(r, fmax(my_rc, src[k]));
        const double sc = w != 0.0 ? o.gm * w / (r2 * r) : 0.0;
        ax += sc * dx; ay += sc * dy; az += sc * dz;
    }
    S->part[s][0][i] = ax; S->part[s][1][i] = ay; S->part[s][2][i] = az;
}

// ---- stage 3: the slices of body i, in slice order (fixed order: the result does not depend on the schedule)
__global__ void __launch_bounds__(NA_THREADS) k_na_sum(const NaScratch *S, int n, double *a)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double ax = 0.0, ay = 0.0, az = 0.0;
    for (int s = 0; s < NA_SLICES; ++s) { ax += S->part[s][0][i]; ay += S->part[s][1][i]; az += S->part[s][2][i]; }
    a[i] = ax; a[n + i] = ay; a[2 * n + i] = az;
}

// ---- the device address of the scratch array, once per device
static std::mutex g_na_mutex;
static NaScratch *g_na_ptr[64] = {};
static thread_local char g_na_err[256] = "";

static int na_scratch_ptr(NaScratch **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= 64) {
        snprintf(g_na_err, sizeof g_na_err, "cudaGetDevice: %s (device %d)", cudaGetErrorString(e), dev);
        return GENGA_ECUDA;
    }
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_ptr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_na_scratch);      // the current device is `dev`: its copy of the array
        if (e != cudaSuccess || !p) {
            snprintf(g_na_err, sizeof g_na_err, "cudaGetSymbolAddress(g_na_scratch) on device %d: %s", dev, cudaGetErrorString(e));
            return GENGA_ECUDA;
        }
        g_na_ptr[dev] = static_cast<NaScratch *>(p);
    }
    *out = g_na_ptr[dev];
    return GENGA_OK;
}

}  // namespace genga

using namespace genga;

extern "C" __attribute__((visibility("default"))) int genga_kick_accel_noalloc(void *stream, int64_t n, double G, const double *m, const double *x,
                                                                                const double *rcrit, double *a)
{
    g_na_err[0] = 0;
    if (n < 0 || !(G > 0.0) || (n > 0 && (!m || !x || !rcrit || !a))) {
        snprintf(g_na_err, sizeof g_na_err, "genga_kick_accel_noalloc: n < 0, G <= 0 or a NULL pointer");
        return GENGA_EINVAL;
    }
    if (n > NA_MAXN) {
        snprintf(g_na_err, sizeof g_na_err, "genga_kick_accel_noalloc: n = %lld exceeds GENGA_NOALLOC_MAX_BODIES = %d (the static scratch array holds no more)",
                 (long long)n, NA_MAXN);
        return GENGA_EINVAL;
    }
    if (n == 0) return GENGA_OK;
    NaScratch *S = nullptr;
    const int r = na_scratch_ptr(&S);
    if (r != GENGA_OK) return r;
    cudaStream_t st = (cudaStream_t)stream;
    const int nb = (int)((n + NA_THREADS - 1) / NA_THREADS);
    k_na_pack<<<nb, NA_THREADS, 0, st>>>(S, (int)n, G, m, x, rcrit);
    k_na_pairs<<<dim3(nb, NA_SLICES), NA_THREADS, 0, st>>>(S, (int)n);
    k_na_sum<<<nb, NA_THREADS, 0, st>>>(S, (int)n, a);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(g_na_err, sizeof g_na_err, "genga_kick_accel_noalloc: launch: %s", cudaGetErrorString(e));
        return GENGA_ECUDA;
    }
    return GENGA_OK;
}

extern "C" __attribute__((visibility("default"))) const char *genga_noalloc_last_error(void) { return g_na_err; }
