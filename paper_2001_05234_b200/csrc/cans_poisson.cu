// cans_poisson.cu -- the C ABI of include/cans_poisson.h: plan creation (tables), the z-solve and
// gradient-correction kernels, and the launch sequences of cans_poisson_solve / cans_projection.
//
// Hot path (eqs. 2b, 5, 6, 2c), default launch sequence:
//   a1+a2  xw_kernel<fwd, DIV> / x_pass_kernel          divergence fused into the forward x transform
//   a3     yt_kernel<fwd> / y_pass_kernel               forward y transform (strided; tiles staged in shared memory, by TMA for 512, 768, 1024)
//   a4     z_solve_kernel                               Thomas solve per (kx, ky) mode (TMA tiles), singular mode pinned, cyclic for periodic z
//   a5     yt_kernel<inv> / y_pass_kernel
//   a6     xw_kernel<inv> / x_pass_kernel
//   a7     grad_correct_kernel (+ face_correct_kernel)  u -= dt G Phi, optionally p_acc += Phi (eq. 2d); then chkdt_kernel on request
// (xw / yt: warp-level 2-pass register FFTs for lengths 512, 768, 1024; x_pass / y_pass: 3-pass shared-memory
//  FFTs for the other lengths.)
// Every x / y / correction kernel takes a range of k-planes (XYArgs::k0, nk; GradArgs::k0, k1); the entry points launch each
// once over all planes -- per-batch launches through L2 were measured and are slower (profiles/r02a_plane_batching.md).
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/cans_poisson.h"
#include "../../include/cans_poisson_probe.h"
#include "plan_tables.hpp"
#include "xy_kernels.cuh"
#include "z_kernels.cuh"
#include "grad_pass.cuh"
#include "chkdt_pass.cuh"
#include "xw_kernels.cuh"
#include "yt_kernels.cuh"
#include "probes.cuh"
#include "errors.hpp"

namespace cans {

static thread_local std::string g_err;
static thread_local int g_status = CANS_OK;

static int fail(int code, const std::string& msg) {
    g_status = code;
    g_err = msg;
    return code;
}
static int fail_cuda(cudaError_t e, const char* where) {
    return fail(CANS_ERR_CUDA, std::string(where) + ": " + cudaGetErrorString(e));
}
// the same for the other translation units (errors.hpp)
void report_ok() { g_status = CANS_OK; }
int report_failure(int code, const char* message) { return fail(code, message); }
int report_cuda_failure(cudaError_t e, const char* where) { return fail_cuda(e, where); }

// ------------------------------------------------------------------------------------------------
// a7: velocity correction u -= dt G Phi (eq. 2c).  A thread owns one pair of x-adjacent cells of a row
// and marches up GRAD_KC planes, carrying Phi(k+1) in registers to become the centre value of the next
// plane: every Phi value is read from HBM once (the row above comes from L2, it is the neighbour thread's
// carry), so the kernel moves its algorithmic 56 B/cell.  The CTAs resident at one time sweep the planes
// together, which keeps the seven streams (Phi, u, v, w in; u, v, w out) sequential in DRAM.
// ------------------------------------------------------------------------------------------------
constexpr int GRAD_KC = 32;

template <bool LAP>
__global__ void __launch_bounds__(256) grad_correct_kernel(const GradArgs a) {
    const int hx = a.nx / 2;
    const size_t cols = (size_t)hx * a.ny;
    const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= cols) return;
    const int k0 = a.k0 + (int)blockIdx.y * GRAD_KC;
    const int k1 = (k0 + GRAD_KC < a.k1) ? k0 + GRAD_KC : a.k1;
    const int i = 2 * (int)(c % hx);
    const int j = (int)(c / hx);
    const size_t plane = (size_t)a.nx * a.ny;
    const size_t rowo = (size_t)j * a.nx + i;
    size_t o = (size_t)k0 * plane + rowo;
    double2 ph = *reinterpret_cast<const double2*>(a.phi + o);
    double2 phm = ph;                              // LAP: the plane below, carried like the centre value
    if (LAP) {
        if (k0 > 0) phm = *reinterpret_cast<const double2*>(a.phi + o - plane);
        else {
            phm = *reinterpret_cast<const double2*>(a.phi + (size_t)a.lz_idx * plane + rowo);
            phm.x *= a.lz_sgn; phm.y *= a.lz_sgn;
        }
    }
    for (int k = k0; k < k1; ++k, o += plane) {
        GradIn in;
        in.o = o;
        in.k = k;
        in.ph = ph;
        if (LAP) {
            in.phzm = phm;
            phm = ph;
            in.phxm = (i > 0) ? a.phi[o - 1] : a.lx_sgn * a.phi[o + a.lx_idx];
            if (j > 0) in.phym = *reinterpret_cast<const double2*>(a.phi + o - a.nx);
            else {
                in.phym = *reinterpret_cast<const double2*>(a.phi + (size_t)k * plane + (size_t)a.ly_idx * a.nx + i);
                in.phym.x *= a.ly_sgn; in.phym.y *= a.ly_sgn;
            }
        }
        in.phx = (i + 2 < a.nx) ? a.phi[o + 2] : a.gx_sgn * a.phi[o - i + a.gx_idx];
        if (j + 1 < a.ny) in.phy = *reinterpret_cast<const double2*>(a.phi + o + a.nx);
        else {
            in.phy = *reinterpret_cast<const double2*>(a.phi + (size_t)k * plane + (size_t)a.gy_idx * a.nx + i);
            in.phy.x *= a.gy_sgn; in.phy.y *= a.gy_sgn;
        }
        if (k + 1 < a.nz) {
            in.phz = *reinterpret_cast<const double2*>(a.phi + o + plane);
            ph = in.phz;                       // centre value of the next plane
        } else {
            in.phz = *reinterpret_cast<const double2*>(a.phi + (size_t)a.gz_idx * plane + rowo);
            in.phz.x *= a.gz_sgn; in.phz.y *= a.gz_sgn;
        }
        in.uu = *reinterpret_cast<const double2*>(a.u + o);
        in.vv = *reinterpret_cast<const double2*>(a.v + o);
        in.ww = *reinterpret_cast<const double2*>(a.w + o);
        if (LAP || a.pacc) in.pa = *reinterpret_cast<const double2*>(a.pacc + o);
        grad_apply<LAP>(a, in);
    }
}

// chkdt (Listing 1): see chkdt_pass.cuh.  One thread per pair of x-adjacent cells, marching up CHK_KC planes.
// Everything that depends on the boundary rule but not on k -- which row a neighbour row is (inside, wrapped, a lower-face
// plane, or absent = 0), where the value beyond the thread's pair comes from at a row end or a warp edge -- is resolved
// ONCE per thread into pointers and strides (ChkStream); the plane loop then only advances pointers.  The step whose k+1
// plane lies beyond the top of the field is peeled off (it runs the general loaders of chkdt_pass.cuh).
constexpr int CHK_KC = 32;

struct ChkStream {
    const double* p;        // the thread's pair (x0, x0 + 1) of the row at the current plane, or NULL: the row reads as 0
    const double* e;        // the value beyond the pair where the neighbouring lane cannot supply it, or NULL (0 / not needed)
};                          // (strides per plane: the field's plane, except for lower-face planes -- kept by the caller)
// u-type rows need u(i-1): from lane - 1, except at lane 0 / i = 0
__device__ __forceinline__ ChkStream chk_stream_u(const ChkArgs& a, int i, int jj, int kk, int lane) {
    ChkStream s = {nullptr, nullptr};
    if (jj >= a.ny) { if (!a.wrap_y) return s; jj = 0; }
    const double* row = a.u + ((size_t)kk * a.ny + jj) * a.nx;
    s.p = row + i;
    if (i > 0) { if (lane == 0) s.e = row + i - 1; }
    else if (a.wrap_x) s.e = row + a.nx - 1;
    else if (a.fx) s.e = a.fx + (size_t)kk * a.ny + jj;       // (stride ny per plane: ChkArgs-dependent, see ue_stride)
    return s;
}
// v / w-type rows need the value at i+2: from lane + 1, except at lane 31 / the row end
__device__ __forceinline__ ChkStream chk_stream_row(const double* row, int i, int nx, int wrap_x, int lane) {
    ChkStream s = {nullptr, nullptr};
    if (!row) return s;
    s.p = row + i;
    if (i + 2 < nx) { if (lane == 31) s.e = row + i + 2; }
    else if (wrap_x) s.e = row;
    return s;
}
__device__ __forceinline__ RowLoad chk_fetch(const ChkStream& s) {
    RowLoad r;
    r.t = s.p ? *reinterpret_cast<const double2*>(s.p) : make_double2(0.0, 0.0);
    r.edge = s.e ? *s.e : 0.0;
    return r;
}
__device__ __forceinline__ void chk_advance(ChkStream& s, long ps, long es) {
    if (s.p) s.p += ps;
    if (s.e) s.e += es;
}

__global__ void __launch_bounds__(256, 2) chkdt_kernel(const ChkArgs a) {
    const int hx = a.nx / 2;
    const size_t cols = (size_t)hx * a.ny;                 // a multiple of 32: a warp is valid as a whole
    const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    double m = 0.0;
    if (c < cols) {
        const int i = 2 * (int)(c % hx);
        const int j = (int)(c / hx);
        const int k0 = (int)blockIdx.y * CHK_KC;
        const int k1 = (k0 + CHK_KC < a.nz) ? k0 + CHK_KC : a.nz;
        const long plane = (long)a.nx * a.ny;
        // carried rows: u(i-1..i+1, j, k); v(i..i+2, j-1 and j, k); w(i..i+2, j, k-1); w(i, i+1; j+1, k-1)
        Row3 uj, vm, vj, wlj, wlp;
        {
            const RowLoad l0 = chk_load_u(a, i, j, k0, lane), l1 = chk_load_v(a, i, j - 1, k0, lane);
            const RowLoad l2 = chk_load_v(a, i, j, k0, lane), l3 = chk_load_w(a, i, j, k0 - 1, lane);
            const RowLoad l4 = chk_load_w(a, i, j + 1, k0 - 1, lane);
            uj = chk_left(l0, i, lane);
            vm = chk_right(l1, i, a.nx, lane); vj = chk_right(l2, i, a.nx, lane);
            wlj = chk_right(l3, i, a.nx, lane); wlp = chk_right(l4, i, a.nx, lane);
        }
        // the six rows fetched per step, positioned at the first step: u(j+1, k), u(j, k+1), v(j-1, k+1), v(j, k+1), w(j, k), w(j+1, k)
        const int kfast = (k1 < a.nz) ? k1 : a.nz - 1;     // steps [k0, kfast) have their k+1 plane inside the field
        // Fast path (warp-uniform): every neighbour row of this warp is a stored row (inside or wrapped) and every value
        // beyond a lane's pair is a stored value -- one running offset and four per-thread deltas address everything.
        // Only when a warp lies inside one row (nx/2 a multiple of 32): then j and the row ends are the same for all its
        // lanes, the branch is warp-uniform (it contains shuffles) and lanes 0 / 31 are the only ones whose outer value the
        // neighbouring lane cannot supply.  Narrower rows take the general loaders, which test i itself.
        const int i_first = i - 2 * lane;
        const bool fast = (hx % 32 == 0) && (a.wrap_y || (j > 0 && j + 1 < a.ny)) &&
                          (a.wrap_x || (i_first > 0 && i_first + 64 < a.nx));
        if (fast) {
            const long d_up = (j + 1 < a.ny) ? (long)a.nx : -(long)(a.ny - 1) * a.nx;      // row j+1 (or row 0)
            const long d_vm = (j > 0) ? -(long)a.nx : (long)(a.ny - 1) * a.nx;             // row j-1 (or row ny-1)
            const long dl = (i > 0) ? -1 : (long)a.nx - 1;                                  // u(i-1), for lane 0
            const long dr = (i + 2 < a.nx) ? 2 : 2 - (long)a.nx;                            // value at i+2, for lane 31
            size_t o = ((size_t)k0 * a.ny + j) * a.nx + i;
            const bool l0 = lane == 0, l31 = lane == 31;
#pragma unroll 2                                    // (two steps per trip: the carried rows rotate by renaming, not by moves)
            for (int k = k0; k < kfast; ++k, o += plane) {
                RowLoad lup, lun, lvm, lvj, lwj, lwp;
                lup.t = *reinterpret_cast<const double2*>(a.u + o + d_up);
                lun.t = *reinterpret_cast<const double2*>(a.u + o + plane);
                lvm.t = *reinterpret_cast<const double2*>(a.v + o + plane + d_vm);
                lvj.t = *reinterpret_cast<const double2*>(a.v + o + plane);
                lwj.t = *reinterpret_cast<const double2*>(a.w + o);
                lwp.t = *reinterpret_cast<const double2*>(a.w + o + d_up);
                lup.edge = lun.edge = lvm.edge = lvj.edge = lwj.edge = lwp.edge = 0.0;
                if (l0) { lup.edge = a.u[o + d_up + dl]; lun.edge = a.u[o + plane + dl]; }
                if (l31) {
                    lvm.edge = a.v[o + plane + d_vm + dr]; lvj.edge = a.v[o + plane + dr];
                    lwj.edge = a.w[o + dr]; lwp.edge = a.w[o + d_up + dr];
                }
                const Row3 up = chk_left(lup, 1, lane), un = chk_left(lun, 1, lane);          // (edge taken at lane 0 / 31 only)
                const Row3 vmn = chk_right(lvm, 0, a.nx, lane), vjn = chk_right(lvj, 0, a.nx, lane);
                const Row3 wj = chk_right(lwj, 0, a.nx, lane), wp = chk_right(lwp, 0, a.nx, lane);
                m = fmax(m, chk_cell_max(a, k, uj, up, un, vm, vj, vmn, vjn, wlj, wlp, wj, wp));
                uj = un; vm = vmn; vj = vjn; wlj = wj; wlp = wp;
            }
        } else {
            ChkStream s_up, s_un, s_vmn, s_vjn, s_wj, s_wp;
            long vstride = plane;                               // v(j-1) is the lower-face plane fy (stride nx) at j = 0 of a wall
            const long ue_stride = (i == 0 && !a.wrap_x && a.fx) ? a.ny : plane;    // u(i-1) from the lower-face plane fx
            if (k0 < kfast) {
                s_up = chk_stream_u(a, i, j + 1, k0, lane);
                s_un = chk_stream_u(a, i, j, k0 + 1, lane);
                const double* vrow = nullptr;
                if (j > 0) vrow = a.v + ((size_t)(k0 + 1) * a.ny + j - 1) * a.nx;
                else if (a.wrap_y) vrow = a.v + ((size_t)(k0 + 1) * a.ny + a.ny - 1) * a.nx;
                else if (a.fy) { vrow = a.fy + (size_t)(k0 + 1) * a.nx; vstride = a.nx; }
                s_vmn = chk_stream_row(vrow, i, a.nx, a.wrap_x, lane);
                s_vjn = chk_stream_row(a.v + ((size_t)(k0 + 1) * a.ny + j) * a.nx, i, a.nx, a.wrap_x, lane);
                s_wj = chk_stream_row(a.w + ((size_t)k0 * a.ny + j) * a.nx, i, a.nx, a.wrap_x, lane);
                const double* wrow = nullptr;
                if (j + 1 < a.ny) wrow = a.w + ((size_t)k0 * a.ny + j + 1) * a.nx;
                else if (a.wrap_y) wrow = a.w + (size_t)k0 * a.ny * a.nx;
                s_wp = chk_stream_row(wrow, i, a.nx, a.wrap_x, lane);
            }
            for (int k = k0; k < kfast; ++k) {
                // all six rows of this step in flight before the first is consumed
                const RowLoad lup = chk_fetch(s_up), lun = chk_fetch(s_un), lvm = chk_fetch(s_vmn), lvj = chk_fetch(s_vjn);
                const RowLoad lwj = chk_fetch(s_wj), lwp = chk_fetch(s_wp);
                chk_advance(s_up, plane, ue_stride); chk_advance(s_un, plane, ue_stride); chk_advance(s_vmn, vstride, vstride);
                chk_advance(s_vjn, plane, plane); chk_advance(s_wj, plane, plane); chk_advance(s_wp, plane, plane);
                const Row3 up = chk_left(lup, i, lane), un = chk_left(lun, i, lane);
                const Row3 vmn = chk_right(lvm, i, a.nx, lane), vjn = chk_right(lvj, i, a.nx, lane);
                const Row3 wj = chk_right(lwj, i, a.nx, lane), wp = chk_right(lwp, i, a.nx, lane);
                m = fmax(m, chk_cell_max(a, k, uj, up, un, vm, vj, vmn, vjn, wlj, wlp, wj, wp));
                uj = un; vm = vmn; vj = vjn; wlj = wj; wlp = wp;
            }
        }
        for (int k = kfast; k < k1; ++k) {                 // (at most) the top plane: its k+1 rows wrap or read as 0
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
    // CTA maximum, then one atomic per CTA -- and only if it can raise the global value (non-negative doubles order
    // like their bit patterns)
    __shared__ double s_max[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) s_max[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int q = 1; q < 8; ++q) m = fmax(m, s_max[q]);
        const unsigned long long bits = (unsigned long long)__double_as_longlong(m);
        if (bits > *reinterpret_cast<volatile unsigned long long*>(a.dti)) atomicMax(a.dti, bits);
    }
}

// Lower boundary face of a direction with a pressure-Dirichlet lower side: the face velocity is an unknown of the
// projection and takes the correction of eq. 2c with the anti-mirrored ghost, face -= dt (Phi_0 - (-Phi_0)) / h.
// Generic over the direction: the plane has n0 x n1 entries (n0 fastest), Phi_0 of entry (a0, a1) sits at
// phi[a0 * s0 + a1 * s1].
struct FaceArgs {
    double* face;
    const double* phi;
    int n0, n1;
    size_t s0, s1;
    double dt, h;
};

__global__ void __launch_bounds__(256) face_correct_kernel(const FaceArgs a) {
    const size_t n = (size_t)a.n0 * a.n1;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x) {
        const size_t a1 = t / a.n0, a0 = t - a1 * a.n0;
        const double first = a.phi[a0 * a.s0 + a1 * a.s1];
        a.face[t] -= a.dt * (first + first) / a.h;
    }
}

}  // namespace cans

using namespace cans;

// ------------------------------------------------------------------------------------------------
// the plan
// ------------------------------------------------------------------------------------------------
constexpr int MAX_REC = CANS_MAX_KERNEL_RECORDS;

struct cans_poisson_plan {
    int nx, ny, nz;
    double lx, ly, lz;
    char bc[3][2];
    int kind_x, kind_y;
    int singular;
    int stagger;              // -1: cell-centred unknown; 0, 1, 2: the unknown lives on the faces of that direction (eq. 3b)
    int nz_solve;             // rows of the tridiagonal systems (nz, or nz - 1 for a face-located unknown between walls)
    // Pivot tables of the z solve (segment-start pivots rstart, singular-column pivots r00), one set per Helmholtz shift
    // alpha: slot 0 is built at plan creation for alpha = 0, the others on the first solve with a new alpha.  An RK3 loop
    // has three gamma_k, so four slots hold everything a plan meets; a fifth alpha replaces the slot used longest ago.
    struct PivotSlot { double alpha; double* rstart; double* r00; unsigned long long last_use; };
    PivotSlot pivots[CANS_MAX_PIVOT_TABLES];
    int npivots;              // slots allocated so far
    unsigned long long pivot_clock;
    int cyclic;               // z periodic: cyclic tridiagonal systems (z_pass.cuh)
    double a0w, cw;           // their wrap couplings
    int nseg, nzp;
    int device;               // the device the plan was created on (tables, kernel attributes)
    int num_sms;
    int z_grid;               // persistent grid of the z solve
    size_t z_smem;
    unsigned int* sched;      // scheduler state (z tile ticket), zeroed at the start of every call
    size_t sched_bytes;
    std::vector<void*> dev_allocs;
    // device tables
    double *lamx, *lamy, *az, *bz, *cz, *gz, *rdzf, *dzf, *rdzc;
    cplx *tw_x, *tw_y, *wpost_x, *wpost_y, *wpre_x, *wpre_y;
    cplx wstep_x[32], wstep_y[32];   // mixed pairs, warp-level kernels: wpre[32 m] (XYArgs::wstep)
    cplx* tw2_x;              // W_nx^(p k1), [nx/32][32]: warp-per-line x kernels (xw_pass.cuh), or NULL
    int use_xw;               // 1: x transforms run the warp-per-line kernels
    cplx* tw2_y;              // the same for ny (yt_pass.cuh), or NULL
    int use_yt;               // 1: y transforms run the persistent TMA-fed kernels (yt_pass.cuh)
    // TMA descriptors of the field the last call worked on: encoded on the host only when the pointer changes
    const double* tmap_field;
    CUtensorMap tmap_y, tmap_z;
    double inv_lz;
    double* face[3];          // registered lower-face planes (caller-owned device memory) or NULL
    double dzc0;              // dzc[0]: distance from the lower z face's ghost centre to the first centre
    // device buffers for the *_host entry points (lazily allocated)
    double* hostbuf[4];
    // optional timing (cans_plan_set_profiling): an event pair around every kernel launch
    int prof;
    int nrec;
    cudaEvent_t ev[2 * MAX_REC];
    const char* kname[MAX_REC];
};

// bracket one kernel launch with events when profiling is on
struct LaunchScope {
    cans_poisson_plan* pl;
    cudaStream_t st;
    bool on;
    LaunchScope(cans_poisson_plan* p, cudaStream_t s, const char* name)
        : pl(p), st(s), on(p->prof && p->nrec < MAX_REC) {
        if (on) { pl->kname[pl->nrec] = name; cudaEventRecord(pl->ev[2 * pl->nrec], st); }
    }
    ~LaunchScope() {
        if (on) { cudaEventRecord(pl->ev[2 * pl->nrec + 1], st); pl->nrec++; }
    }
};

static int kind_of(char lo, char up, int* kind) {
    if (lo == 'P' && up == 'P') { *kind = KIND_PP; return CANS_OK; }
    if (lo == 'N' && up == 'N') { *kind = KIND_NN; return CANS_OK; }
    if (lo == 'D' && up == 'D') { *kind = KIND_DD; return CANS_OK; }
    if (lo == 'N' && up == 'D') { *kind = KIND_ND; return CANS_OK; }
    if (lo == 'D' && up == 'N') { *kind = KIND_DN; return CANS_OK; }
    return CANS_ERR_INVALID_ARG;
}

template <class T>
static cudaError_t upload(cans_poisson_plan* pl, const std::vector<double>& h, T** dptr) {
    void* d = nullptr;
    cudaError_t e = cudaMalloc(&d, h.size() * sizeof(double));
    if (e != cudaSuccess) return e;
    pl->dev_allocs.push_back(d);
    e = cudaMemcpy(d, h.data(), h.size() * sizeof(double), cudaMemcpyHostToDevice);
    *dptr = reinterpret_cast<T*>(d);
    return e;
}

// layout of the scheduler state (unsigned ints)
enum { SCHED_Z_TICKET = 0, SCHED_WORDS = 8 };

static ZArgs make_zargs(const cans_poisson_plan* pl, double* p, double alpha = 0.0, int slot = 0) {
    ZArgs z;
    z.alpha = alpha;
    z.nz_solve = pl->nz_solve;
    z.nx = pl->nx; z.ny = pl->ny; z.nz = pl->nz;
    z.nseg = pl->nseg;
    z.ncols = (long)pl->nx * pl->ny;
    z.p = p;
    z.lamx = pl->lamx; z.lamy = pl->lamy;
    z.az = pl->az; z.bz = pl->bz; z.cz = pl->cz; z.gz = pl->gz;
    z.rstart = pl->pivots[slot].rstart;
    z.scale = 1.0 / ((double)pl->nx * (double)pl->ny);
    z.singular = pl->singular && alpha == 0.0;
    z.r00 = pl->pivots[slot].r00;
    z.dzf = pl->dzf;
    z.inv_lz = pl->inv_lz;
    const int tc = z_tc_for(pl->nseg);
    z.ntiles = (z.ncols + tc - 1) / tc;
    z.ticket = pl->sched + SCHED_Z_TICKET;
    z.cyclic = pl->cyclic; z.a0w = pl->a0w; z.cw = pl->cw;
    return z;
}

static XYArgs make_xyargs(const cans_poisson_plan* pl, double* p, bool xdir) {
    XYArgs a;
    std::memset(&a, 0, sizeof(a));
    a.nx = pl->nx; a.ny = pl->ny; a.nz = pl->nz;
    a.k0 = 0; a.nk = pl->nz;
    a.kind = xdir ? pl->kind_x : pl->kind_y;
    a.tw = xdir ? pl->tw_x : pl->tw_y;
    a.wpost = xdir ? pl->wpost_x : pl->wpost_y;
    a.wpre = xdir ? pl->wpre_x : pl->wpre_y;
    std::memcpy(a.wstep, xdir ? pl->wstep_x : pl->wstep_y, sizeof(a.wstep));
    a.p = p;
    return a;
}

// one more pivot-table slot for the shift alpha (contents are filled by z_setup_launch)
static cudaError_t alloc_pivot_slot(cans_poisson_plan* pl, double alpha) {
    void *d0 = nullptr, *d1 = nullptr;
    cudaError_t e = cudaMalloc(&d0, sizeof(double) * (size_t)pl->nseg * pl->nx * pl->ny);
    if (e != cudaSuccess) return e;
    e = cudaMalloc(&d1, sizeof(double) * (size_t)pl->nz);
    if (e != cudaSuccess) { cudaFree(d0); return e; }
    pl->dev_allocs.push_back(d0);
    pl->dev_allocs.push_back(d1);
    cans_poisson_plan::PivotSlot& sl = pl->pivots[pl->npivots++];
    sl.alpha = alpha; sl.rstart = (double*)d0; sl.r00 = (double*)d1; sl.last_use = 0;
    return cudaSuccess;
}

static const char* const XY_NAMES[5] = {"x_fwd", "x_fwd_div", "x_inv", "y_fwd", "y_inv"};

// one x / y transform launch over the planes [a.k0, a.k0 + a.nk)
static int launch_xy_any(cans_poisson_plan* pl, int n, int op, const XYArgs& a, cudaStream_t st) {
    cudaError_t err = cudaSuccess;
    const bool xdir = (op == OP_X_FWD || op == OP_X_FWD_DIV || op == OP_X_INV);
    LaunchScope scope(pl, st, XY_NAMES[op]);
    bool done = false;
    if (xdir && pl->use_xw) done = xw_launch(n, op, a, pl->tw2_x, st, &err);
    else if (!xdir && pl->use_yt) done = yt_launch(n, op, a, pl->tw2_y, &pl->tmap_y, pl->num_sms, st, &err);
    if (!done)
        done = launch_xy_group_a(n, op, a, st, &err) || launch_xy_group_b(n, op, a, st, &err) ||
               launch_xy_group_c(n, op, a, st, &err) || launch_xy_group_d(n, op, a, st, &err);
    if (!done) return fail(CANS_ERR_UNSUPPORTED_SIZE, "transform length not instantiated");
    if (err != cudaSuccess) return fail_cuda(err, xdir ? "x transform launch" : "y transform launch");
    return CANS_OK;
}

// plan time: dynamic shared memory opt-in of every transform kernel this plan can run, on the plan's device
static cudaError_t configure_kernels(cans_poisson_plan* pl) {
    const XYArgs dummy = make_xyargs(pl, nullptr, true);
    cudaError_t e = cudaSuccess;
    const int lens[2] = {pl->nx, pl->ny};
    for (int n : lens) {
        const bool found = launch_xy_group_a(n, OP_CONFIGURE, dummy, 0, &e) || launch_xy_group_b(n, OP_CONFIGURE, dummy, 0, &e) ||
                           launch_xy_group_c(n, OP_CONFIGURE, dummy, 0, &e) || launch_xy_group_d(n, OP_CONFIGURE, dummy, 0, &e);
        if (!found) return cudaErrorInvalidValue;
        if (e != cudaSuccess) return e;
    }
    if (pl->use_xw) { xw_launch(pl->nx, OP_CONFIGURE, dummy, pl->tw2_x, 0, &e); if (e != cudaSuccess) return e; }
    if (pl->use_yt) { yt_launch(pl->ny, OP_CONFIGURE, dummy, pl->tw2_y, nullptr, pl->num_sms, 0, &e); if (e != cudaSuccess) return e; }
    return e;
}

extern "C" {

const char* cans_last_error(void) { return g_err.c_str(); }
int cans_last_status(void) { return g_status; }
const char* cans_version(void) { return "0.2"; }

void cans_poisson_plan_destroy(cans_poisson_plan* plan) {
    if (!plan) return;
    for (void* d : plan->dev_allocs) cudaFree(d);
    for (int i = 0; i < 4; ++i) if (plan->hostbuf[i]) cudaFree(plan->hostbuf[i]);
    if (plan->prof) for (int i = 0; i < 2 * MAX_REC; ++i) cudaEventDestroy(plan->ev[i]);
    delete plan;
}

cans_poisson_plan* cans_poisson_plan_create(int nx, int ny, int nz, double lx, double ly, double lz,
                                            const char bc[3][2], const double* dzc, const double* dzf) {
    return cans_helmholtz_plan_create(nx, ny, nz, lx, ly, lz, bc, dzc, dzf, -1);
}

cans_poisson_plan* cans_helmholtz_plan_create(int nx, int ny, int nz, double lx, double ly, double lz,
                                              const char bc[3][2], const double* dzc, const double* dzf, int stagger) {
    g_status = CANS_OK;
    g_err.clear();
    if (!bc) { fail(CANS_ERR_INVALID_ARG, "bc is NULL"); return nullptr; }
    if (nx < 2 || ny < 2 || nz < 2) { fail(CANS_ERR_INVALID_ARG, "nx, ny, nz must be >= 2"); return nullptr; }
    if (!(lx > 0.0) || !(ly > 0.0) || !(lz > 0.0)) { fail(CANS_ERR_INVALID_ARG, "lx, ly, lz must be > 0"); return nullptr; }
    if ((dzc == nullptr) != (dzf == nullptr)) { fail(CANS_ERR_INVALID_ARG, "dzc and dzf must both be given or both be NULL"); return nullptr; }
    for (int d = 0; d < 3; ++d)
        for (int s = 0; s < 2; ++s) {
            const char ch = bc[d][s];
            if (ch != 'P' && ch != 'N' && ch != 'D') { fail(CANS_ERR_INVALID_ARG, "bc letters must be 'P', 'N' or 'D'"); return nullptr; }
        }
    for (int d = 0; d < 3; ++d)
        if ((bc[d][0] == 'P') != (bc[d][1] == 'P')) { fail(CANS_ERR_INVALID_ARG, "periodic boundaries must be two-sided"); return nullptr; }
    int kx, ky;
    if (kind_of(bc[0][0], bc[0][1], &kx) != CANS_OK || kind_of(bc[1][0], bc[1][1], &ky) != CANS_OK) {
        fail(CANS_ERR_INVALID_ARG, "unknown boundary pair");
        return nullptr;
    }
    if (stagger < -1 || stagger > 2) { fail(CANS_ERR_INVALID_ARG, "stagger must be -1, 0, 1 or 2"); return nullptr; }
    if ((stagger == 0 || stagger == 1) && bc[stagger][0] != 'P') {
        fail(CANS_ERR_UNSUPPORTED_BC, "an unknown on the faces of a non-periodic x or y direction needs the node-based DST-I / DCT-I transforms (not implemented)");
        return nullptr;
    }
    if (stagger == 2 && bc[2][0] == 'N') {
        fail(CANS_ERR_UNSUPPORTED_BC, "an unknown on the z faces with a lower 'N' side is not implemented (the lower boundary "
                                      "face would be an unknown and the compact layout has no slot for it): use 'P', ('D','D') or ('D','N')");
        return nullptr;
    }
    FftRadices fx, fy;
    if (!fft_lookup(nx, &fx) || !fft_lookup(ny, &fy)) {
        fail(CANS_ERR_UNSUPPORTED_SIZE, "nx and ny must be one of 16,32,48,64,96,128,192,256,384,512,768,1024,1536,2048");
        return nullptr;
    }
    const int nseg = (nz + Z_MROWS - 1) / Z_MROWS;
    if (nseg > 64) { fail(CANS_ERR_UNSUPPORTED_SIZE, "nz too large for the z-solve tiling (max 1024)"); return nullptr; }
    if (z_solve_smem_bytes(nseg) > Z_SMEM_LIMIT) {
        fail(CANS_ERR_UNSUPPORTED_SIZE, "nz too large for the z-solve tiling (shared memory)");
        return nullptr;
    }
    std::vector<double> hdzc(nz + 1), hdzf(nz);
    for (int k = 0; k < nz; ++k) hdzf[k] = dzf ? dzf[k] : lz / nz;
    for (int k = 0; k <= nz; ++k) hdzc[k] = dzc ? dzc[k] : lz / nz;
    for (int k = 0; k < nz; ++k) if (!(hdzf[k] > 0.0)) { fail(CANS_ERR_INVALID_ARG, "dzf must be positive"); return nullptr; }
    for (int k = 0; k <= nz; ++k) if (!(hdzc[k] > 0.0)) { fail(CANS_ERR_INVALID_ARG, "dzc must be positive"); return nullptr; }
    if (bc[2][0] == 'P' && std::fabs(hdzc[0] - hdzc[nz]) > 1e-12 * (hdzc[0] + hdzc[nz])) {
        // dzc[0] and dzc[nz] are the same distance (last centre to first centre through the wrap): two values would give a
        // gradient and a divergence that do not compose to the Laplacian, i.e. a projection that is not divergence free
        fail(CANS_ERR_INVALID_ARG, "periodic z needs a single-valued wrap spacing: dzc[0] == dzc[nz]");
        return nullptr;
    }

    cans_poisson_plan* pl = new (std::nothrow) cans_poisson_plan();
    if (!pl) { fail(CANS_ERR_ALLOC, "host allocation failed"); return nullptr; }
    pl->nx = nx; pl->ny = ny; pl->nz = nz; pl->lx = lx; pl->ly = ly; pl->lz = lz;
    std::memcpy(pl->bc, bc, 6);
    pl->kind_x = kx; pl->kind_y = ky;
    pl->nseg = nseg; pl->nzp = nseg * Z_MROWS;
    for (int i = 0; i < 4; ++i) pl->hostbuf[i] = nullptr;
    for (int i = 0; i < 3; ++i) pl->face[i] = nullptr;
    pl->dzc0 = hdzc[0];
    pl->prof = 0; pl->nrec = 0;
    pl->tmap_field = nullptr;
    pl->singular = (kx == KIND_PP || kx == KIND_NN) && (ky == KIND_PP || ky == KIND_NN) && bc[2][0] != 'D' && bc[2][1] != 'D';
    pl->cyclic = bc[2][0] == 'P';
    pl->stagger = stagger;
    pl->nz_solve = (stagger == 2 && bc[2][0] == 'D' && bc[2][1] == 'D') ? nz - 1 : nz;
    pl->npivots = 0;
    pl->pivot_clock = 0;
    pl->device = 0;
    cudaGetDevice(&pl->device);
    pl->num_sms = 148;
    cudaDeviceGetAttribute(&pl->num_sms, cudaDevAttrMultiProcessorCount, pl->device);

    const double dx = lx / nx, dy = ly / ny;
    ZRows zr = make_z_rows(nz, pl->nzp, hdzc.data(), hdzf.data(), bc[2][0], bc[2][1], stagger == 2);
    pl->inv_lz = 1.0 / zr.lz_sum;
    pl->a0w = zr.a0w; pl->cw = zr.cw;
    std::vector<double> rdzc(nz);
    for (int k = 0; k < nz; ++k) rdzc[k] = 1.0 / hdzc[k + 1];

    cudaError_t e = cudaSuccess;
    auto up = [&](const std::vector<double>& h, auto** d) { if (e == cudaSuccess) e = upload(pl, h, d); };
    up(make_lambda_positions(nx, kx, dx), &pl->lamx);
    up(make_lambda_positions(ny, ky, dy), &pl->lamy);
    up(zr.a, &pl->az); up(zr.b, &pl->bz); up(zr.c, &pl->cz); up(zr.g, &pl->gz);
    up(zr.rdzf, &pl->rdzf); up(zr.dzf, &pl->dzf); up(rdzc, &pl->rdzc);
    up(make_pass_twiddles(fx), &pl->tw_x);
    up(make_pass_twiddles(fy), &pl->tw_y);
    up(kind_mixed(kx) ? make_post_twiddles_mixed(nx) : make_post_twiddles(nx), &pl->wpost_x);
    up(kind_mixed(ky) ? make_post_twiddles_mixed(ny) : make_post_twiddles(ny), &pl->wpost_y);
    pl->wpre_x = pl->wpre_y = nullptr;
    std::memset(pl->wstep_x, 0, sizeof(pl->wstep_x));
    std::memset(pl->wstep_y, 0, sizeof(pl->wstep_y));
    auto steps = [](const std::vector<double>& wpre, int n, cplx* out) {
        for (int m = 0; m < 32 && 32 * m < n; ++m) out[m] = make_double2(wpre[2 * (32 * m)], wpre[2 * (32 * m) + 1]);
    };
    if (kind_mixed(kx)) { const std::vector<double> h = make_pre_twiddles_mixed(nx); steps(h, nx, pl->wstep_x); up(h, &pl->wpre_x); }
    if (kind_mixed(ky)) { const std::vector<double> h = make_pre_twiddles_mixed(ny); steps(h, ny, pl->wstep_y); up(h, &pl->wpre_y); }
    pl->tw2_x = nullptr;
    pl->use_xw = 0;
    if (xw_supported(nx)) {
        up(make_two_pass_twiddles(nx), &pl->tw2_x);
        pl->use_xw = 1;
    }
    pl->tw2_y = nullptr;
    pl->use_yt = 0;
    if (yt_supported(ny) && (nx / 2) % YT_COLS == 0) {
        up(make_two_pass_twiddles(ny), &pl->tw2_y);
        pl->use_yt = 1;
    }
    if (e == cudaSuccess) e = alloc_pivot_slot(pl, 0.0);
    if (e == cudaSuccess) {
        pl->sched_bytes = sizeof(unsigned int) * SCHED_WORDS;
        void* d = nullptr;
        e = cudaMalloc(&d, pl->sched_bytes);
        if (e == cudaSuccess) { pl->dev_allocs.push_back(d); pl->sched = (unsigned int*)d; e = cudaMemset(d, 0, pl->sched_bytes); }
    }
    if (e == cudaSuccess) {
        ZArgs z = make_zargs(pl, nullptr);
        e = z_setup_launch(z, pl->pivots[0].rstart, pl->pivots[0].r00, 0);
        if (e == cudaSuccess) e = cudaDeviceSynchronize();
    }
    if (e == cudaSuccess) e = z_solve_configure(nseg, pl->cyclic, pl->num_sms, &pl->z_grid, &pl->z_smem);
    if (e == cudaSuccess) e = configure_kernels(pl);
    if (e != cudaSuccess) {
        const std::string msg = std::string("plan creation: ") + cudaGetErrorString(e);
        const int code = (e == cudaErrorMemoryAllocation) ? CANS_ERR_ALLOC : CANS_ERR_CUDA;
        cans_poisson_plan_destroy(pl);
        cudaGetLastError();
        fail(code, msg);
        return nullptr;
    }
    return pl;
}

static int launch_z(cans_poisson_plan* pl, double* p, double alpha, cudaStream_t st) {
    int slot = -1;
    for (int i = 0; i < pl->npivots; ++i)
        if (pl->pivots[i].alpha == alpha) slot = i;
    const bool build = slot < 0;
    if (build) {
        // a shift this plan has not met (or has dropped): take a free slot -- the only allocation a solve can make, at most
        // CANS_MAX_PIVOT_TABLES - 1 times in the life of a plan -- or, when all are taken or the board is full, the slot
        // used longest ago (never slot 0: the Poisson table)
        if (pl->npivots < CANS_MAX_PIVOT_TABLES && alloc_pivot_slot(pl, alpha) == cudaSuccess) slot = pl->npivots - 1;
        else {
            cudaGetLastError();
            if (pl->npivots < 2) slot = 0;
            else {
                slot = 1;
                for (int i = 2; i < pl->npivots; ++i)
                    if (pl->pivots[i].last_use < pl->pivots[slot].last_use) slot = i;
            }
            pl->pivots[slot].alpha = alpha;
        }
    }
    pl->pivots[slot].last_use = ++pl->pivot_clock;
    ZArgs z = make_zargs(pl, p, alpha, slot);
    if (build) {
        // the segment-start pivots depend on the shift: fill the table on this stream (one sweep per column, no field
        // data: ~N/16 doubles written) before the solve that uses it; stream order also protects a replaced slot
        LaunchScope scope(pl, st, "z_setup");
        cudaError_t e = z_setup_launch(z, pl->pivots[slot].rstart, pl->pivots[slot].r00, st);
        if (e != cudaSuccess) { pl->pivots[slot].alpha = NAN; return fail_cuda(e, "z pivot table launch"); }
    }
    LaunchScope scope(pl, st, "z_solve");
    cudaError_t e = z_solve_launch(z, pl->z_grid, pl->z_smem, &pl->tmap_z, st);
    if (e != cudaSuccess) return fail_cuda(e, "z solve launch");
    return CANS_OK;
}

static int launch_grad(cans_poisson_plan* pl, const GradArgs& g, cudaStream_t st) {
    const size_t cols = (size_t)pl->nx / 2 * pl->ny;
    dim3 grid((unsigned)((cols + 255) / 256), (unsigned)((g.k1 - g.k0 + GRAD_KC - 1) / GRAD_KC));
    LaunchScope scope(pl, st, "grad_correct");
    if (g.pacc && g.lap_coef != 0.0) grad_correct_kernel<true><<<grid, 256, 0, st>>>(g);     // eq. 3e
    else grad_correct_kernel<false><<<grid, 256, 0, st>>>(g);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(e, "gradient correction launch");
    return CANS_OK;
}

// TMA descriptors of the field: host-side encode only when the caller passes another buffer than last time
static int ensure_tensor_maps(cans_poisson_plan* pl, double* p) {
    if (pl->tmap_field == p) return CANS_OK;
    cudaError_t e = z_make_tensor_map(&pl->tmap_z, p, (long)pl->nx * pl->ny, pl->nz, pl->nseg);
    if (e == cudaSuccess && pl->use_yt) e = yt_make_tensor_map(&pl->tmap_y, p, pl->nx, pl->ny, pl->nz);
    if (e != cudaSuccess) { pl->tmap_field = nullptr; return fail_cuda(e, "tensor map encode"); }
    pl->tmap_field = p;
    return CANS_OK;
}

// the whole path shared by both entry points; `divargs` selects the fused-divergence load (a1),
// `grad` the velocity correction (a7)
static int run_core(cans_poisson_plan* pl, double* p, const XYArgs* divargs, const GradArgs* grad, cudaStream_t st,
                    double alpha = 0.0) {
    int rc;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != pl->device)
        return fail(CANS_ERR_INVALID_ARG, "the plan was created on another device than the current one");
    pl->nrec = 0;
    cudaError_t me = cudaMemsetAsync(pl->sched, 0, pl->sched_bytes, st);
    if (me != cudaSuccess) return fail_cuda(me, "scheduler reset");
    if ((rc = ensure_tensor_maps(pl, p))) return rc;
    const XYArgs ax = make_xyargs(pl, p, true), ay = make_xyargs(pl, p, false);
    if (divargs) rc = launch_xy_any(pl, pl->nx, OP_X_FWD_DIV, *divargs, st);      // a1 + a2
    else rc = launch_xy_any(pl, pl->nx, OP_X_FWD, ax, st);                          // a2
    if (rc) return rc;
    if ((rc = launch_xy_any(pl, pl->ny, OP_Y_FWD, ay, st))) return rc;              // a3
    if ((rc = launch_z(pl, p, alpha, st))) return rc;                               // a4
    if ((rc = launch_xy_any(pl, pl->ny, OP_Y_INV, ay, st))) return rc;              // a5
    if ((rc = launch_xy_any(pl, pl->nx, OP_X_INV, ax, st))) return rc;              // a6
    if (grad) return launch_grad(pl, *grad, st);                                    // a7
    return CANS_OK;
}

int cans_plan_launches_per_solve(const cans_poisson_plan*) { return 5; }
int cans_plan_launches_per_projection(const cans_poisson_plan* plan) {
    int n = 6;
    if (plan)
        for (int d = 0; d < 3; ++d) n += (plan->bc[d][0] == 'D' && plan->face[d]) ? 1 : 0;   // lower-face corrections
    return n;
}

int cans_poisson_solve(cans_poisson_plan* plan, double* p, void* stream) {
    g_status = CANS_OK;
    if (!plan || !p) return fail(CANS_ERR_INVALID_ARG, "plan and p must be non-NULL");
    if ((reinterpret_cast<size_t>(p) & 15) != 0) return fail(CANS_ERR_INVALID_ARG, "p must be 16-byte aligned");
    if (plan->stagger == 2) return fail(CANS_ERR_INVALID_ARG, "a plan for an unknown on the z faces solves cans_helmholtz_solve only");
    return run_core(plan, p, nullptr, nullptr, (cudaStream_t)stream);
}

int cans_helmholtz_solve(cans_poisson_plan* plan, double* q, double alpha, void* stream) {
    g_status = CANS_OK;
    if (!plan || !q) return fail(CANS_ERR_INVALID_ARG, "plan and q must be non-NULL");
    if ((reinterpret_cast<size_t>(q) & 15) != 0) return fail(CANS_ERR_INVALID_ARG, "q must be 16-byte aligned");
    if (!(alpha < 0.0)) return fail(CANS_ERR_INVALID_ARG, "alpha must be < 0 (eq. 3b: alpha = -2/(gamma nu dt))");
    return run_core(plan, q, nullptr, nullptr, (cudaStream_t)stream, alpha);
}

static int chkdt_enqueue(cans_poisson_plan* plan, const double* u, const double* v, const double* w, double* dti, cudaStream_t st);

int cans_chkdt(cans_poisson_plan* plan, const double* u, const double* v, const double* w, double* dti, void* stream) {
    g_status = CANS_OK;
    if (!plan) return fail(CANS_ERR_INVALID_ARG, "plan is NULL");
    plan->nrec = 0;
    return chkdt_enqueue(plan, u, v, w, dti, (cudaStream_t)stream);
}

static int chkdt_enqueue(cans_poisson_plan* plan, const double* u, const double* v, const double* w, double* dti, cudaStream_t st) {
    if (!u || !v || !w || !dti) return fail(CANS_ERR_INVALID_ARG, "u, v, w, dti must be non-NULL");
    if (((reinterpret_cast<size_t>(u) | reinterpret_cast<size_t>(v) | reinterpret_cast<size_t>(w)) & 15) != 0 ||
        (reinterpret_cast<size_t>(dti) & 7) != 0)
        return fail(CANS_ERR_INVALID_ARG, "fields must be 16-byte aligned, dti 8-byte aligned");
    for (int d = 0; d < 3; ++d)
        if (plan->bc[d][0] == 'D' && !plan->face[d])
            return fail(CANS_ERR_NEEDS_FACE, "a lower 'D' side needs a lower-face plane (cans_projection_set_lower_face)");
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != plan->device)
        return fail(CANS_ERR_INVALID_ARG, "the plan was created on another device than the current one");
    ChkArgs c;
    c.nx = plan->nx; c.ny = plan->ny; c.nz = plan->nz;
    c.u = u; c.v = v; c.w = w;
    c.fx = plan->face[0]; c.fy = plan->face[1]; c.fz = plan->face[2];
    c.wrap_x = plan->bc[0][0] == 'P'; c.wrap_y = plan->bc[1][0] == 'P'; c.wrap_z = plan->bc[2][0] == 'P';
    c.rdx = (double)plan->nx / plan->lx; c.rdy = (double)plan->ny / plan->ly;
    c.rdzf = plan->rdzf; c.rdzc = plan->rdzc;
    c.dti = reinterpret_cast<unsigned long long*>(dti);
    cudaError_t e = cudaMemsetAsync(dti, 0, sizeof(double), st);
    if (e != cudaSuccess) return fail_cuda(e, "dti reset");
    const size_t cols = (size_t)plan->nx / 2 * plan->ny;
    dim3 grid((unsigned)((cols + 255) / 256), (unsigned)((plan->nz + CHK_KC - 1) / CHK_KC));
    LaunchScope scope(plan, st, "chkdt");
    chkdt_kernel<<<grid, 256, 0, st>>>(c);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(e, "chkdt launch");
    return CANS_OK;
}

int cans_projection(cans_poisson_plan* plan, double* u, double* v, double* w, double* p, double dt, void* stream) {
    return cans_projection_step(plan, u, v, w, p, nullptr, dt, nullptr, stream);
}

int cans_projection_step(cans_poisson_plan* plan, double* u, double* v, double* w, double* p, double* p_acc, double dt,
                         double* dti, void* stream) {
    return cans_projection_step_implicit(plan, u, v, w, p, p_acc, dt, 0.0, dti, stream);
}

int cans_projection_step_implicit(cans_poisson_plan* plan, double* u, double* v, double* w, double* p, double* p_acc, double dt,
                                  double nu_dt_half, double* dti, void* stream) {
    g_status = CANS_OK;
    if (!(nu_dt_half >= 0.0)) return fail(CANS_ERR_INVALID_ARG, "nu_dt_half (gamma nu dt / 2 of eq. 3e) must be >= 0");
    if (nu_dt_half > 0.0 && !p_acc) return fail(CANS_ERR_INVALID_ARG, "eq. 3e updates p_acc: it must be non-NULL when nu_dt_half > 0");
    if (!plan || !u || !v || !w || !p) return fail(CANS_ERR_INVALID_ARG, "plan, u, v, w, p must be non-NULL");
    if (plan->stagger == 2) return fail(CANS_ERR_INVALID_ARG, "a plan for an unknown on the z faces solves cans_helmholtz_solve only");
    if (p_acc && ((reinterpret_cast<size_t>(p_acc) & 15) != 0 || p_acc == p || p_acc == u || p_acc == v || p_acc == w))
        return fail(CANS_ERR_INVALID_ARG, "p_acc must be 16-byte aligned and distinct from p, u, v, w");
    if (p == u || p == v || p == w || u == v || u == w || v == w)
        return fail(CANS_ERR_INVALID_ARG, "u, v, w, p must be four distinct arrays (p is overwritten while u, v, w are still read)");
    if (!(dt > 0.0)) return fail(CANS_ERR_INVALID_ARG, "dt must be > 0");
    if (((reinterpret_cast<size_t>(p) | reinterpret_cast<size_t>(u) | reinterpret_cast<size_t>(v) |
          reinterpret_cast<size_t>(w)) & 15) != 0)
        return fail(CANS_ERR_INVALID_ARG, "fields must be 16-byte aligned");
    for (int d = 0; d < 3; ++d)
        if (plan->bc[d][0] == 'D' && !plan->face[d])
            return fail(CANS_ERR_NEEDS_FACE, "a lower 'D' side needs a lower-face plane (cans_projection_set_lower_face)");
    cudaStream_t st = (cudaStream_t)stream;
    XYArgs a = make_xyargs(plan, p, true);
    a.u = u; a.v = v; a.w = w;
    a.rdzf = plan->rdzf;
    a.rdx = (double)plan->nx / plan->lx;
    a.rdy = (double)plan->ny / plan->ly;
    a.rdt = 1.0 / dt;
    a.wrap_x = plan->bc[0][0] == 'P';
    a.wrap_y = plan->bc[1][0] == 'P';
    a.wrap_z = plan->bc[2][0] == 'P';
    a.fx = plan->face[0]; a.fy = plan->face[1]; a.fz = plan->face[2];
    GradArgs g;
    g.nx = plan->nx; g.ny = plan->ny; g.nz = plan->nz;
    g.k0 = 0; g.k1 = plan->nz;
    g.u = u; g.v = v; g.w = w; g.phi = p;
    g.pacc = p_acc;
    g.rdzc = plan->rdzc;
    g.dt = dt;
    g.dt_rdx = dt * a.rdx;
    g.dt_rdy = dt * a.rdy;
    auto ghost = [](char up, int n, int* idx, double* sgn) {
        if (up == 'P') { *idx = 0; *sgn = 1.0; }
        else if (up == 'N') { *idx = n - 1; *sgn = 1.0; }
        else { *idx = n - 1; *sgn = -1.0; }
    };
    ghost(plan->bc[0][1], plan->nx, &g.gx_idx, &g.gx_sgn);
    ghost(plan->bc[1][1], plan->ny, &g.gy_idx, &g.gy_sgn);
    ghost(plan->bc[2][1], plan->nz, &g.gz_idx, &g.gz_sgn);
    auto ghost_below = [](char lo, int n, int* idx, double* sgn) {
        if (lo == 'P') { *idx = n - 1; *sgn = 1.0; }
        else if (lo == 'N') { *idx = 0; *sgn = 1.0; }
        else { *idx = 0; *sgn = -1.0; }
    };
    ghost_below(plan->bc[0][0], plan->nx, &g.lx_idx, &g.lx_sgn);
    ghost_below(plan->bc[1][0], plan->ny, &g.ly_idx, &g.ly_sgn);
    ghost_below(plan->bc[2][0], plan->nz, &g.lz_idx, &g.lz_sgn);
    g.lap_coef = nu_dt_half;
    g.rdx2 = a.rdx * a.rdx; g.rdy2 = a.rdy * a.rdy;
    g.rdzc0 = 1.0 / plan->dzc0;
    g.rdzf = plan->rdzf;
    int rc = run_core(plan, p, &a, &g, st);
    if (rc) return rc;
    // a7 on the registered lower faces of pressure-Dirichlet sides (planes on 'N' sides are prescribed inflow)
    const int nx = plan->nx, ny = plan->ny, nz = plan->nz;
    for (int d = 0; d < 3; ++d) {
        if (plan->bc[d][0] != 'D') continue;
        FaceArgs fa;
        fa.face = plan->face[d];
        fa.phi = p;
        fa.dt = dt;
        if (d == 0) { fa.n0 = ny; fa.n1 = nz; fa.s0 = (size_t)nx; fa.s1 = (size_t)nx * ny; fa.h = plan->lx / nx; }
        else if (d == 1) { fa.n0 = nx; fa.n1 = nz; fa.s0 = 1; fa.s1 = (size_t)nx * ny; fa.h = plan->ly / ny; }
        else { fa.n0 = nx; fa.n1 = ny; fa.s0 = 1; fa.s1 = (size_t)nx; fa.h = plan->dzc0; }
        const size_t n = (size_t)fa.n0 * fa.n1;
        LaunchScope scope(plan, st, "face_correct");
        face_correct_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(fa);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return fail_cuda(e, "lower-face correction launch");
    }
    if (dti) {
        // chkdt on the corrected velocities: its own kernel -- the face averages need the corrected values of the
        // neighbouring threads' cells, which an in-place correction cannot provide race-free
        rc = chkdt_enqueue(plan, u, v, w, dti, (cudaStream_t)stream);
        if (rc) return rc;
    }
    return CANS_OK;
}

int cans_probe_fp64_fma(double* fma_per_s, void* stream) {
    g_status = CANS_OK;
    if (!fma_per_s) return fail(CANS_ERR_INVALID_ARG, "fma_per_s is NULL");
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaError_t e = probe_fp64_fma(sms, fma_per_s, (cudaStream_t)stream);
    if (e != cudaSuccess) return fail_cuda(e, "FP64 FMA probe");
    return CANS_OK;
}

int cans_probe_tile_copy(cans_poisson_plan* plan, double* p, int which, float* ms, void* stream) {
    g_status = CANS_OK;
    if (!plan || !p || !ms) return fail(CANS_ERR_INVALID_ARG, "NULL argument");
    if ((reinterpret_cast<size_t>(p) & 15) != 0) return fail(CANS_ERR_INVALID_ARG, "p must be 16-byte aligned");
    int rc = ensure_tensor_maps(plan, p);
    if (rc) return rc;
    TileCopyShape sh;
    const CUtensorMap* tmap;
    CUtensorMap tmap_wide;
    if (which == 0) {            // z solve: tiles of z_tc_for(nseg) columns x nz rows of the (nz, nx*ny) view
        const int tc = z_tc_for(plan->nseg);
        sh.ntiles = ((long)plan->nx * plan->ny + tc - 1) / tc; sh.m0 = sh.ntiles; sh.s0 = tc; sh.s1 = 0;
        z_boxes(plan->nseg, &sh.nbox, &sh.box_rows); sh.box_cols = tc;
        tmap = &plan->tmap_z;
    } else if (which == 1) {     // TMA-fed y transforms: tiles of 16 doubles x ny rows of one k-plane
        if (!plan->use_yt || plan->ny > 768) return fail(CANS_ERR_UNSUPPORTED_SIZE, "the y-tile probe needs two tile buffers: ny = 512, 768");
        sh.m0 = plan->nx / 2 / YT_COLS; sh.ntiles = sh.m0 * plan->nz; sh.s0 = 2 * YT_COLS; sh.s1 = plan->ny;
        sh.box_rows = YT_BOX_ROWS; sh.nbox = plan->ny / YT_BOX_ROWS; sh.box_cols = 2 * YT_COLS;
        tmap = &plan->tmap_y;
    } else if (which == 2) {     // the z view again, row segments twice as wide: tiles of 32 columns x 256 rows (two per column tile)
        const long ncols = (long)plan->nx * plan->ny;
        cudaError_t te = make_tensor_map_2d(&tmap_wide, p, (unsigned long long)ncols, (unsigned long long)plan->nz,
                                            (unsigned long long)ncols * sizeof(double), 32, 256, CU_TENSOR_MAP_SWIZZLE_NONE);
        if (te != cudaSuccess) return fail_cuda(te, "tensor map encode");
        sh.m0 = (ncols + 31) / 32; sh.ntiles = sh.m0 * ((plan->nz + 255) / 256); sh.s0 = 32; sh.s1 = 256;
        sh.box_rows = 256; sh.nbox = 1; sh.box_cols = 32;
        tmap = &tmap_wide;
    } else {
        return fail(CANS_ERR_INVALID_ARG, "which must be 0 (z tiles), 1 (y tiles) or 2 (z view, 32-column tiles)");
    }
    cudaError_t e = probe_tile_copy(tmap, sh, plan->num_sms, ms, (cudaStream_t)stream);
    if (e != cudaSuccess) return fail_cuda(e, "tile copy probe");
    return CANS_OK;
}

int cans_plan_set_profiling(cans_poisson_plan* plan, int enable) {
    g_status = CANS_OK;
    if (!plan) return fail(CANS_ERR_INVALID_ARG, "plan is NULL");
    if (enable && !plan->prof) {
        for (int i = 0; i < 2 * MAX_REC; ++i) {
            cudaError_t e = cudaEventCreate(&plan->ev[i]);
            if (e != cudaSuccess) return fail_cuda(e, "cudaEventCreate");
        }
        plan->prof = 1;
    } else if (!enable && plan->prof) {
        for (int i = 0; i < 2 * MAX_REC; ++i) cudaEventDestroy(plan->ev[i]);
        plan->prof = 0;
    }
    plan->nrec = 0;
    return CANS_OK;
}

int cans_plan_kernel_times(cans_poisson_plan* plan, float* ms, int capacity) {
    g_status = CANS_OK;
    if (!plan || !ms) { fail(CANS_ERR_INVALID_ARG, "NULL argument"); return -1; }
    if (!plan->prof) { fail(CANS_ERR_INVALID_ARG, "profiling is not enabled"); return -1; }
    int n = plan->nrec < capacity ? plan->nrec : capacity;
    for (int i = 0; i < n; ++i) {
        cudaError_t e = cudaEventSynchronize(plan->ev[2 * i + 1]);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms[i], plan->ev[2 * i], plan->ev[2 * i + 1]);
        if (e != cudaSuccess) { fail_cuda(e, "kernel timing"); return -1; }
    }
    return n;
}

const char* cans_plan_kernel_name(const cans_poisson_plan* plan, int idx) {
    if (!plan || idx < 0 || idx >= plan->nrec) return "";
    return plan->kname[idx];
}

int cans_projection_set_lower_face(cans_poisson_plan* plan, int dir, double* face_plane) {
    g_status = CANS_OK;
    if (!plan || dir < 0 || dir > 2) return fail(CANS_ERR_INVALID_ARG, "bad plan or direction");
    if (face_plane) {
        if (plan->bc[dir][0] == 'P')
            return fail(CANS_ERR_INVALID_ARG, "a periodic direction has no lower boundary face (it is the wrapped value)");
        if ((reinterpret_cast<size_t>(face_plane) & 15) != 0)
            return fail(CANS_ERR_INVALID_ARG, "the face plane must be 16-byte aligned");
    }
    plan->face[dir] = face_plane;
    return CANS_OK;
}

static int ensure_hostbufs(cans_poisson_plan* pl, int count) {
    const size_t bytes = sizeof(double) * (size_t)pl->nx * pl->ny * pl->nz;
    for (int i = 0; i < count; ++i)
        if (!pl->hostbuf[i]) {
            cudaError_t e = cudaMalloc((void**)&pl->hostbuf[i], bytes);
            if (e != cudaSuccess) { cudaGetLastError(); return fail(CANS_ERR_ALLOC, "device buffer for host entry point"); }
        }
    return CANS_OK;
}

int cans_poisson_solve_host(cans_poisson_plan* plan, double* p_host, void* stream) {
    g_status = CANS_OK;
    if (!plan || !p_host) return fail(CANS_ERR_INVALID_ARG, "plan and p_host must be non-NULL");
    int rc = ensure_hostbufs(plan, 1);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = sizeof(double) * (size_t)plan->nx * plan->ny * plan->nz;
    cudaError_t e = cudaMemcpyAsync(plan->hostbuf[0], p_host, bytes, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return fail_cuda(e, "H2D copy");
    if ((rc = cans_poisson_solve(plan, plan->hostbuf[0], stream))) return rc;
    e = cudaMemcpyAsync(p_host, plan->hostbuf[0], bytes, cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) return fail_cuda(e, "D2H copy");
    e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fail_cuda(e, "stream synchronize");
    return CANS_OK;
}

int cans_projection_host(cans_poisson_plan* plan, double* u_host, double* v_host, double* w_host,
                         double* p_host, double dt, void* stream) {
    g_status = CANS_OK;
    if (!plan || !u_host || !v_host || !w_host || !p_host) return fail(CANS_ERR_INVALID_ARG, "NULL argument");
    int rc = ensure_hostbufs(plan, 4);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = sizeof(double) * (size_t)plan->nx * plan->ny * plan->nz;
    double* hsrc[3] = {u_host, v_host, w_host};
    cudaError_t e;
    for (int i = 0; i < 3; ++i) {
        e = cudaMemcpyAsync(plan->hostbuf[i], hsrc[i], bytes, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return fail_cuda(e, "H2D copy");
    }
    if ((rc = cans_projection(plan, plan->hostbuf[0], plan->hostbuf[1], plan->hostbuf[2], plan->hostbuf[3], dt, stream))) return rc;
    double* hdst[4] = {u_host, v_host, w_host, p_host};
    for (int i = 0; i < 4; ++i) {
        e = cudaMemcpyAsync(hdst[i], plan->hostbuf[i], bytes, cudaMemcpyDeviceToHost, st);
        if (e != cudaSuccess) return fail_cuda(e, "D2H copy");
    }
    e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fail_cuda(e, "stream synchronize");
    return CANS_OK;
}

}  // extern "C"
