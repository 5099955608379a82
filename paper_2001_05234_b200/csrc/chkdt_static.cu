// chkdt_static.cu -- cans_chkdt_static: the reduction of Listing 1 (eq. 4) for callers that cannot
// allocate device memory.
//
// Who that is.  Everything else in this library hangs off a plan, and a plan is built with cudaMalloc (its tables) and
// released with cudaFree.  A solver that sized its own arena to fill the 180 GB of the board has nothing left for the driver
// to hand out; a time loop that runs several streams cannot afford cudaMalloc / cudaFree either, because both wait for the
// whole device and so serialise everything in flight.  Such a caller still wants the stable time step of its velocity
// field.  This entry point takes no plan and calls nothing that allocates: what the kernel needs besides the caller's
// arrays -- the reciprocal z spacings the planned kernel reads from plan tables, and one partial maximum per CTA -- lives in
// the file-scope array g_chk_scratch below, which is part of the library image (every GPU that loads the library holds its
// 528 KB until exit).
//
// What follows from one shared array:
//   * sizes are bounded (CANS_STATIC_MAX_NZ, CANS_STATIC_MAX_CTAS); larger ones are refused, not truncated;
//   * the array keeps whatever the previous call left: the prepare kernel rewrites the spacing tables and zeroes the
//     arrival counter at the start of every call, and the partial maxima are all written before they are read;
//   * two calls that run on the GPU at the same time (different streams, or different host threads) would share the tables,
//     the partials and the counter: they race.  Calls on one stream are ordered and safe.
//   * the device address of the array is looked up once per device, on the first call made with that device current
//     (cudaGetSymbolAddress; the name g_chk_scratch in host code is only a handle for that lookup).  Make that first call
//     outside any stream capture.
//
// The arithmetic is the planned kernel's: the loaders and the face sums of chkdt_pass.cuh, every plane through the general
// (boundary-aware) loaders.  A maximum does not depend on the order it is taken in, so the result equals cans_chkdt's bit
// for bit.
#include <cuda_runtime.h>

#include <mutex>

#include "../../include/cans_poisson.h"
#include "chkdt_pass.cuh"
#include "errors.hpp"

namespace cans {

constexpr int CHKS_KC = 32;                                   // planes one CTA marches up
constexpr int CHKS_THREADS = 256;
constexpr int CHKS_OFF_RDZF = 0;                              // [CANS_STATIC_MAX_NZ]   1 / dzf[k]
constexpr int CHKS_OFF_RDZC = CANS_STATIC_MAX_NZ;             // [CANS_STATIC_MAX_NZ]   1 / dzc[k+1]
constexpr int CHKS_OFF_CTAMAX = 2 * CANS_STATIC_MAX_NZ;       // [CANS_STATIC_MAX_CTAS] maximum of each CTA
constexpr int CHKS_OFF_ARRIVED = CHKS_OFF_CTAMAX + CANS_STATIC_MAX_CTAS;   // one word: CTAs that have published theirs
constexpr int CHKS_WORDS = CHKS_OFF_ARRIVED + 32;             // (the counter keeps a 256-byte line to itself)

// The scratch itself.  Device code may name it; host code must go through scratch_address().
static __device__ __align__(256) double g_chk_scratch[CHKS_WORDS];

// spacing tables and counter of the call that is starting (one CTA)
__global__ void __launch_bounds__(CHKS_THREADS) chkdt_static_prepare(double* scr, const double* dzc, const double* dzf, int nz,
                                                                     double dz_uniform) {
    for (int k = threadIdx.x; k < nz; k += blockDim.x) {
        scr[CHKS_OFF_RDZF + k] = 1.0 / (dzf ? dzf[k] : dz_uniform);
        scr[CHKS_OFF_RDZC + k] = 1.0 / (dzc ? dzc[k + 1] : dz_uniform);
    }
    if (threadIdx.x == 0) *reinterpret_cast<unsigned int*>(scr + CHKS_OFF_ARRIVED) = 0u;
}

__global__ void __launch_bounds__(CHKS_THREADS, 2) chkdt_static_kernel(const ChkArgs a, double* scr, double* dti) {
    const int hx = a.nx / 2;
    const size_t cols = (size_t)hx * a.ny;                 // a multiple of 32 (checked by the entry point): whole warps
    const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    double m = 0.0;
    if (c < cols) {
        const int i = 2 * (int)(c % hx);
        const int j = (int)(c / hx);
        const int k0 = (int)blockIdx.y * CHKS_KC;
        const int k1 = (k0 + CHKS_KC < a.nz) ? k0 + CHKS_KC : a.nz;
        // carried rows, as in chkdt_kernel: u(i-1..i+1, j, k); v(i..i+2, j-1 and j, k); w(i..i+2, j and j+1, k-1)
        Row3 uj, vm, vj, wlj, wlp;
        {
            const RowLoad l0 = chk_load_u(a, i, j, k0, lane), l1 = chk_load_v(a, i, j - 1, k0, lane);
            const RowLoad l2 = chk_load_v(a, i, j, k0, lane), l3 = chk_load_w(a, i, j, k0 - 1, lane);
            const RowLoad l4 = chk_load_w(a, i, j + 1, k0 - 1, lane);
            uj = chk_left(l0, i, lane);
            vm = chk_right(l1, i, a.nx, lane); vj = chk_right(l2, i, a.nx, lane);
            wlj = chk_right(l3, i, a.nx, lane); wlp = chk_right(l4, i, a.nx, lane);
        }
        for (int k = k0; k < k1; ++k) {
            const RowLoad lup = chk_load_u(a, i, j + 1, k, lane);
            const RowLoad lun = chk_load_u(a, i, j, k + 1, lane);
            const RowLoad lvm = chk_load_v(a, i, j - 1, k + 1, lane), lvj = chk_load_v(a, i, j, k + 1, lane);
            const RowLoad lwj = chk_load_w(a, i, j, k, lane), lwp = chk_load_w(a, i, j + 1, k, lane);
            const Row3 up = chk_left(lup, i, lane), un = chk_left(lun, i, lane);
            const Row3 vmn = chk_right(lvm, i, a.nx, lane), vjn = chk_right(lvj, i, a.nx, lane);
            const Row3 wj = chk_right(lwj, i, a.nx, lane), wp = chk_right(lwp, i, a.nx, lane);
            m = fmax(m, chk_cell_max(a, k, uj, up, un, vm, vj, vmn, vjn, wlj, wlp, wj, wp));
            uj = un; vm = vmn; vj = vjn; wlj = wj; wlp = wp;
        }
    }
    // CTA maximum into the scratch; the CTA that arrives last folds all of them into dti
    __shared__ double s_max[CHKS_THREADS / 32];
    __shared__ bool s_last;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if (lane == 0) s_max[threadIdx.x >> 5] = m;
    __syncthreads();
    const unsigned int nctas = gridDim.x * gridDim.y;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int q = 1; q < CHKS_THREADS / 32; ++q) m = fmax(m, s_max[q]);
        scr[CHKS_OFF_CTAMAX + blockIdx.y * gridDim.x + blockIdx.x] = m;
        __threadfence();                                   // the maximum is visible before the arrival is
        const unsigned int before = atomicAdd(reinterpret_cast<unsigned int*>(scr + CHKS_OFF_ARRIVED), 1u);
        s_last = (before + 1 == nctas);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double t = 0.0;
    for (unsigned int q = threadIdx.x; q < nctas; q += CHKS_THREADS) t = fmax(t, __ldcg(scr + CHKS_OFF_CTAMAX + q));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t = fmax(t, __shfl_xor_sync(0xffffffffu, t, o));
    __syncthreads();                                       // (s_max is reused)
    if (lane == 0) s_max[threadIdx.x >> 5] = t;
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int q = 1; q < CHKS_THREADS / 32; ++q) t = fmax(t, s_max[q]);
        *dti = t;
    }
}

// Device address of g_chk_scratch on the current device: looked up on the first call per device, cached afterwards.
constexpr int CHKS_MAX_DEVICES = 64;
static std::mutex g_scratch_mutex;
static double* g_scratch_addr[CHKS_MAX_DEVICES] = {};

static cudaError_t scratch_address(int dev, double** out) {
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_addr[dev]) {
        void* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_chk_scratch);   // resolves against the CURRENT device (= dev)
        if (e != cudaSuccess) return e;
        g_scratch_addr[dev] = static_cast<double*>(ptr);
    }
    *out = g_scratch_addr[dev];
    return cudaSuccess;
}

}  // namespace cans

using namespace cans;

extern "C" int cans_chkdt_static(int nx, int ny, int nz, double lx, double ly, double lz, const char bc[3][2],
                                 const double* dzc, const double* dzf, const double* u, const double* v, const double* w,
                                 const double* face_x, const double* face_y, const double* face_z, double* dti, void* stream) {
    report_ok();
    if (!bc || !u || !v || !w || !dti) return report_failure(CANS_ERR_INVALID_ARG, "bc, u, v, w, dti must be non-NULL");
    if (nx < 2 || ny < 2 || nz < 2) return report_failure(CANS_ERR_INVALID_ARG, "nx, ny, nz must be >= 2");
    if (!(lx > 0.0) || !(ly > 0.0) || !(lz > 0.0)) return report_failure(CANS_ERR_INVALID_ARG, "lx, ly, lz must be > 0");
    if ((dzc == nullptr) != (dzf == nullptr))
        return report_failure(CANS_ERR_INVALID_ARG, "dzc and dzf must both be given or both be NULL");
    for (int d = 0; d < 3; ++d) {
        for (int s = 0; s < 2; ++s)
            if (bc[d][s] != 'P' && bc[d][s] != 'N' && bc[d][s] != 'D')
                return report_failure(CANS_ERR_INVALID_ARG, "bc letters must be 'P', 'N' or 'D'");
        if ((bc[d][0] == 'P') != (bc[d][1] == 'P'))
            return report_failure(CANS_ERR_INVALID_ARG, "periodic boundaries must be two-sided");
    }
    const double* face[3] = {face_x, face_y, face_z};
    size_t align16 = reinterpret_cast<size_t>(u) | reinterpret_cast<size_t>(v) | reinterpret_cast<size_t>(w);
    for (int d = 0; d < 3; ++d) {
        if (face[d] && bc[d][0] == 'P')
            return report_failure(CANS_ERR_INVALID_ARG, "a periodic direction has no lower boundary face (it is the wrapped value)");
        if (!face[d] && bc[d][0] == 'D')
            return report_failure(CANS_ERR_NEEDS_FACE, "a lower 'D' side needs its lower-face plane");
        align16 |= reinterpret_cast<size_t>(face[d]);
    }
    if ((align16 & 15) != 0 || (reinterpret_cast<size_t>(dti) & 7) != 0)
        return report_failure(CANS_ERR_INVALID_ARG, "fields and face planes must be 16-byte aligned, dti 8-byte aligned");
    if (nx % 2 != 0 || ((size_t)(nx / 2) * ny) % 32 != 0)
        return report_failure(CANS_ERR_UNSUPPORTED_SIZE, "nx must be even and (nx/2)*ny a multiple of 32");
    if (nz > CANS_STATIC_MAX_NZ)
        return report_failure(CANS_ERR_UNSUPPORTED_SIZE, "cans_chkdt_static: nz exceeds CANS_STATIC_MAX_NZ (the static scratch holds 1024 spacings)");
    const size_t cols = (size_t)(nx / 2) * ny;
    const size_t gx = (cols + CHKS_THREADS - 1) / CHKS_THREADS, gy = (size_t)(nz + CHKS_KC - 1) / CHKS_KC;
    if (gx * gy > (size_t)CANS_STATIC_MAX_CTAS)
        return report_failure(CANS_ERR_UNSUPPORTED_SIZE,
                              "cans_chkdt_static: ceil(nx*ny/512) * ceil(nz/32) exceeds CANS_STATIC_MAX_CTAS (the static scratch "
                              "holds one partial maximum per CTA); use cans_chkdt with a plan for larger grids");
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return report_cuda_failure(e, "cudaGetDevice");
    if (dev < 0 || dev >= CHKS_MAX_DEVICES) return report_failure(CANS_ERR_INVALID_ARG, "device ordinal beyond 63");
    double* scr = nullptr;
    if ((e = scratch_address(dev, &scr)) != cudaSuccess) return report_cuda_failure(e, "cudaGetSymbolAddress(g_chk_scratch)");

    ChkArgs c;
    c.nx = nx; c.ny = ny; c.nz = nz;
    c.u = u; c.v = v; c.w = w;
    c.fx = face_x; c.fy = face_y; c.fz = face_z;
    c.wrap_x = bc[0][0] == 'P'; c.wrap_y = bc[1][0] == 'P'; c.wrap_z = bc[2][0] == 'P';
    c.rdx = (double)nx / lx; c.rdy = (double)ny / ly;
    c.rdzf = scr + CHKS_OFF_RDZF; c.rdzc = scr + CHKS_OFF_RDZC;
    c.dti = nullptr;                                       // (the planned kernel's atomic target: not used here)
    cudaStream_t st = (cudaStream_t)stream;
    chkdt_static_prepare<<<1, CHKS_THREADS, 0, st>>>(scr, dzc, dzf, nz, lz / nz);
    if ((e = cudaGetLastError()) != cudaSuccess) return report_cuda_failure(e, "chkdt_static_prepare launch");
    chkdt_static_kernel<<<dim3((unsigned)gx, (unsigned)gy), CHKS_THREADS, 0, st>>>(c, scr, dti);
    if ((e = cudaGetLastError()) != cudaSuccess) return report_cuda_failure(e, "chkdt_static_kernel launch");
    return CANS_OK;
}
