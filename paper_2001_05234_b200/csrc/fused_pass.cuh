// fused_pass.cuh -- passes A and C of the projection as persistent task kernels fused through L2.
//
//   pass A = a1 + a2 + a3 : divergence (eq. 2b) -> forward x transform -> forward y transform
//   pass C = a5 + a6 + a7 : inverse y -> inverse x (eq. 6) -> u -= dt G Phi (eq. 2c)
//
// A k-plane (C5: 6.3 MB) does not fit one SM's shared memory but fits the 126 MB L2 many times, so the
// intermediate of an x/y transform pair never has to reach HBM: CTAs are persistent and draw TICKETS from
// one global counter; the ticket list is ordered plane by plane (host-built `Segment` table), every
// plane has completion counters, and a task waits (acquire) only on counters that are incremented by
// tasks with SMALLER tickets.  Such tasks are either finished or held by a running CTA, so the scheme
// cannot deadlock and needs no co-residency guarantee.  HBM then sees each pass once
// (32 / 64 B per cell for the projection, 16 / 16 for the bare Poisson solve).
//
// HBM latency is hidden with the L2 as the staging buffer: while a CTA works on ticket t it issues
// bulk L2 prefetches (cp.async.bulk.prefetch.L2) for the HBM-resident input rows of ticket t + lookahead.
#pragma once
#include <cuda_runtime.h>
#include "xy_pass.cuh"
#include "grad_pass.cuh"

namespace cans {

enum TaskType : int { TASK_X = 0, TASK_Y = 1, TASK_G = 2 };

// a run of consecutive tickets: `count` tasks of one type on plane k
struct Segment {
    unsigned first, count;
    int type, k;
    int dep0, dep1;             // counters that must reach target0/1 before the task reads its input (-1: none)
    unsigned target0, target1;
    int signal;                 // counter incremented once the task's output is visible (-1: none)
    int pad;
};

struct FusedArgs {
    XYArgs ax, ay;              // x / y direction (ax carries u, v, w and the divergence factors)
    GradArgs g;
    const Segment* segs;        // sorted by `first`; the last entry is a sentinel with count = 0xffffffff
    unsigned total;             // number of tickets
    unsigned lookahead;         // prefetch distance in tickets
    unsigned* ticket;
    unsigned* counters;
    int mode;                   // pass A: 1 = fused divergence; pass C: 1 = gradient tasks present
    int grows;                  // rows per gradient task
};

#if defined(__CUDACC__)
CANS_D unsigned ld_acquire_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}
CANS_D void l2_prefetch_bulk(const void* p, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;\n" ::"l"(p), "r"(bytes) : "memory");
}
// thread 0 spins until the counter reaches its target; the barrier publishes the acquire to the CTA
CANS_D void wait_counter(const unsigned* c, unsigned target) {
    unsigned ns = 32;
    while (ld_acquire_u32(c) < target) {
        __nanosleep(ns);
        if (ns < 512) ns *= 2;
    }
}
#endif

#if defined(__CUDACC__)
extern __shared__ __align__(16) unsigned char cans_dyn_smem[];

template <int A, int B> struct MaxOf { static constexpr int value = A > B ? A : B; };

// INV = false: pass A (X = forward x transform [+ divergence], Y = forward y transform)
// INV = true : pass C (Y = inverse y transform, X = inverse x transform, G = gradient correction)
template <class PX, class PY, int NFX, int TXC, int NT, bool INV>
__global__ void __launch_bounds__(NT, 2) fused_xy_kernel(const FusedArgs a) {
    constexpr int WORK = MaxOf<NFX * PX::NPAD, PY::N * TXC>::value;
    typedef XPass<PX, NFX, NT, WORK> X;
    typedef YPass<PY, TXC, NT, WORK + PX::TW_TOTAL> Y;
    cplx* sm = reinterpret_cast<cplx*>(cans_dyn_smem);
    __shared__ unsigned s_ticket;
    const int tid = threadIdx.x;
    const int nx = a.ax.nx, ny = a.ax.ny;
    const int hp = ny >> 1;
    const int nyt = (nx >> 1) / TXC;
    const size_t rowb = (size_t)nx * sizeof(double);
    X::load_twiddles(a.ax, sm, tid);
    Y::load_twiddles(a.ay, sm, tid);
    int cur = 0, curp = 0;
    while (true) {
        __syncthreads();                               // the previous task is done with smem and s_ticket
        if (tid == 0) s_ticket = atomicAdd(a.ticket, 1u);
        __syncthreads();
        const unsigned t = s_ticket;
        if (t >= a.total) break;

        // ---- L2 prefetch of the HBM-resident input rows of ticket t + lookahead ----
        const unsigned tp = t + a.lookahead;
        if (tp < a.total) {
            while (tp - a.segs[curp].first >= a.segs[curp].count) ++curp;
            const int ptype = a.segs[curp].type;
            const int pk = a.segs[curp].k;
            const int pidx = (int)(tp - a.segs[curp].first);
            if (!INV && ptype == TASK_X) {
                const int j0 = 2 * NFX * pidx;
                const int nr = min(2 * NFX, ny - j0);
                const size_t ro = ((size_t)pk * ny + j0) * (size_t)nx;
                if (a.mode) {
                    if (tid < 3 * nr) {
                        const int fld = tid / nr, r = tid - fld * nr;
                        const double* src = (fld == 0 ? a.ax.u : (fld == 1 ? a.ax.v : a.ax.w)) + ro + (size_t)r * nx;
                        l2_prefetch_bulk(src, (unsigned)rowb);
                    }
                } else if (tid < nr) {
                    l2_prefetch_bulk(a.ax.p + ro + (size_t)tid * nx, (unsigned)rowb);
                }
            } else if (INV && ptype == TASK_Y) {
                const int j0 = (int)(((long)pidx * ny) / nyt);
                const int j1 = (int)(((long)(pidx + 1) * ny) / nyt);
                if (tid < j1 - j0)
                    l2_prefetch_bulk(a.ay.p + ((size_t)pk * ny + j0 + tid) * (size_t)nx, (unsigned)rowb);
            } else if (INV && ptype == TASK_G) {
                const int j0 = pidx * a.grows;
                const int nr = min(a.grows, ny - j0);
                const size_t ro = ((size_t)pk * ny + j0) * (size_t)nx;
                if (tid < 3 * nr) {
                    const int fld = tid / nr, r = tid - fld * nr;
                    const double* src = (fld == 0 ? a.g.u : (fld == 1 ? a.g.v : a.g.w)) + ro + (size_t)r * nx;
                    l2_prefetch_bulk(src, (unsigned)rowb);
                }
            }
        }

        // ---- decode the ticket, wait for the planes it reads ----
        while (t - a.segs[cur].first >= a.segs[cur].count) ++cur;
        const Segment sg = a.segs[cur];
        const int idx = (int)(t - sg.first);
        const int k = sg.k;
        if (sg.dep0 >= 0) {
            if (tid == 0) {
                wait_counter(a.counters + sg.dep0, sg.target0);
                if (sg.dep1 >= 0) wait_counter(a.counters + sg.dep1, sg.target1);
                __threadfence();
            }
            __syncthreads();
        }

        if (sg.type == TASK_X) {
            const long pair0 = (long)k * hp + (long)idx * NFX;
            const long lim = (long)(k + 1) * hp;
            if (!INV) {
                if (a.mode) X::template load_forward<true>(a.ax, sm, pair0, lim, tid);
                else X::template load_forward<false>(a.ax, sm, pair0, lim, tid);
                __syncthreads();
                X::pass1_fwd(sm, tid);
                __syncthreads();
                if (PX::R2 > 1) { X::pass2_fwd(sm, tid); __syncthreads(); }
                X::pass3_fwd(sm, tid);
                __syncthreads();
                X::store_forward(a.ax, sm, pair0, lim, tid);
            } else {
                X::load_inverse(a.ax, sm, pair0, lim, tid);
                __syncthreads();
                X::pass3_inv(sm, tid);
                __syncthreads();
                if (PX::R2 > 1) { X::pass2_inv(sm, tid); __syncthreads(); }
                X::pass1_inv(sm, tid);
                __syncthreads();
                X::store_inverse(a.ax, sm, pair0, lim, tid);
            }
        } else if (sg.type == TASK_Y) {
            if (!INV) {
                Y::load_forward(a.ay, sm, idx, k, tid);
                __syncthreads();
                Y::pass1_fwd(sm, tid);
                __syncthreads();
                if (PY::R2 > 1) { Y::pass2_fwd(sm, tid); __syncthreads(); }
                Y::pass3_fwd(sm, tid);
                __syncthreads();
                Y::store_forward(a.ay, sm, idx, k, tid);
            } else {
                Y::load_inverse(a.ay, sm, idx, k, tid);
                __syncthreads();
                Y::pass3_inv(sm, tid);
                __syncthreads();
                if (PY::R2 > 1) { Y::pass2_inv(sm, tid); __syncthreads(); }
                Y::pass1_inv(sm, tid);
                __syncthreads();
                Y::store_inverse(a.ay, sm, idx, k, tid);
            }
        } else if (INV) {
            const int hx = nx >> 1;
            const int j0 = idx * a.grows;
            const int j1 = min(j0 + a.grows, ny);
            const size_t t0 = ((size_t)k * ny + j0) * (size_t)hx;
            const size_t t1 = ((size_t)k * ny + j1) * (size_t)hx;
            for (size_t tt = t0 + tid; tt < t1; tt += NT) grad_correct_pair(a.g, tt);
        }

        if (sg.signal >= 0) {
            __syncthreads();                           // every thread's stores are issued ...
            if (tid == 0) {
                __threadfence();                       // ... and made visible before the count moves
                atomicAdd(a.counters + sg.signal, 1u);
            }
        }
    }
}

template <class K>
static cudaError_t fused_set_smem(K kern, size_t bytes) {
    return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

// what: 0 = configure (sets *grid, *smem), 1 = launch pass A, 2 = launch pass C
template <class PX, class PY, int NFX, int TXC, int NT>
cudaError_t fused_run(int what, const FusedArgs* a, int num_sms, int* grid, size_t* smem, cudaStream_t st) {
    constexpr int WORK = MaxOf<NFX * PX::NPAD, PY::N * TXC>::value;
    const size_t bytes = sizeof(cplx) * (size_t)(WORK + PX::TW_TOTAL + PY::TW_TOTAL);
    auto ka = fused_xy_kernel<PX, PY, NFX, TXC, NT, false>;
    auto kc = fused_xy_kernel<PX, PY, NFX, TXC, NT, true>;
    if (what == 0) {
        cudaError_t e = fused_set_smem(ka, bytes);
        if (e == cudaSuccess) e = fused_set_smem(kc, bytes);
        if (e != cudaSuccess) return e;
        int oa = 0, oc = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&oa, ka, NT, bytes);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&oc, kc, NT, bytes);
        if (e != cudaSuccess) return e;
        const int occ = oa < oc ? oa : oc;
        if (occ < 1) return cudaErrorLaunchOutOfResources;
        *grid = occ * num_sms;
        *smem = bytes;
        return cudaSuccess;
    }
    if (what == 1) ka<<<(unsigned)*grid, NT, *smem, st>>>(*a);
    else kc<<<(unsigned)*grid, NT, *smem, st>>>(*a);
    return cudaGetLastError();
}
#endif  // __CUDACC__

// tiling of the fused kernels per transform length (host and device agree through these)
constexpr int FUSED_NT = 256;
constexpr int FUSED_GROWS = 8;
inline int fused_nfx(int nx) { return nx <= 384 ? 8 : 4; }          // row pairs per x task
inline int fused_txc(int ny) { return ny <= 512 ? 8 : 4; }          // complex columns per y task
inline bool fused_supported(int nx, int ny) {
    auto ok = [](int n) { return n == 256 || n == 384 || n == 512 || n == 768 || n == 1024; };
    return ok(nx) && ok(ny);
}
// one function per nx (fused_x*.cu); returns false if (nx, ny) is not instantiated
bool fused_dispatch(int nx, int ny, int what, const FusedArgs* a, int num_sms, int* grid, size_t* smem,
                    cudaStream_t st, cudaError_t* err);

}  // namespace cans
