// fused_pass.cuh -- passes A and C of the projection as persistent task kernels fused through L2.
//
//   pass A = a1 + a2 + a3 : divergence (eq. 2b) -> forward x transform -> forward y transform
//   pass C = a5 + a6 + a7 : inverse y -> inverse x (eq. 6) -> u -= dt G Phi (eq. 2c)
//
// A k-plane (C5: 6.3 MB) does not fit one SM's shared memory but fits the 126 MB L2 many times, so the
// intermediate planes of a pass never have to reach HBM.  Persistent CTAs (two per SM) draw TICKETS from a
// global counter.  Tickets are ordered in ROUNDS; round r holds, in this order, the tasks of up to three
// SLOTS, slot s working on plane k = r - off[s]:
//     pass A:  X(r)  [divergence +] x transforms     Y(r-2)  y transforms
//     pass C:  Y(r)  inverse y      X(r-2)  inverse x      G(r-5)  gradient rows   (Poisson only: no G)
// A task of slot s waits until every task of slot s-1 on its plane has signalled (G also waits for the
// plane above, whose Phi it reads).  A task therefore only ever waits for tasks with SMALLER tickets,
// which are finished or held by a running CTA: no deadlock, no co-residency requirement.
// The HBM-resident input rows of the next task are prefetched into L2 (cp.async.bulk.prefetch.L2) while
// the current task runs; the task bodies are the 3-pass phase functions of xy_pass.cuh.
//
// STATUS (round 1): correct and parity-tested, but slower than the unfused sequence (19.9 ms vs 11.9 ms
// per C5 projection): the CTA-synchronous phases serialise on an SM and a plane lag long enough to avoid
// spinning pushes dirty intermediate planes out of L2.  Opt-in through cans_plan_set_fusion; see
// DESIGN.md section 7 for the measurements of the three variants that were tried and the plan
// (warp-level x tasks of xw_pass.cuh inside the persistent kernel).
#pragma once
#include <cuda_runtime.h>
#include "xy_pass.cuh"
#include "grad_pass.cuh"

namespace cans {

enum TaskType : int { TASK_END = -2, TASK_NONE = -1, TASK_X = 0, TASK_Y = 1, TASK_G = 2 };

struct FusedArgs {
    XYArgs ax, ay;              // x / y direction (ax carries u, v, w and the divergence factors)
    GradArgs g;
    int nslots;
    int slot_type[3];
    int slot_off[3];            // plane lag of the slot within a round
    unsigned slot_count[3];     // tasks per plane
    unsigned per_round;         // sum of slot_count
    unsigned total;             // (nz + max off) * per_round
    unsigned* ticket;
    unsigned* counters;         // [slot][cstride]
    int cstride;
    int grows;                  // rows per gradient task
    int mode;                   // pass A: 1 = divergence fused into the x load
};

struct Task { int type, k, idx, slot; };

// tiling of the fused kernels per transform length (host and device agree through these)
constexpr int FUSED_NT = 256;
constexpr int FUSED_GROWS = 8;
// the work buffer of a CTA stays <= 67 KB so that two CTAs (with both twiddle tables each) share an SM
constexpr int fused_nfx(int nx) { return nx >= 512 ? 4 : 8; }        // row pairs per x task
constexpr int fused_txc(int ny) { return ny >= 768 ? 4 : 8; }        // complex columns per y task
inline bool fused_supported(int nx, int ny) {
    auto ok = [](int n) { return n == 256 || n == 384 || n == 512 || n == 768 || n == 1024; };
    return ok(nx) && ok(ny);
}

#if defined(__CUDACC__)
CANS_D unsigned ld_acquire_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}
CANS_D void l2_prefetch_bulk(const void* p, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;\n" ::"l"(p), "r"(bytes) : "memory");
}

CANS_D void wait_counter(const unsigned* c, unsigned target) {
    unsigned ns = 32;
    while (ld_acquire_u32(c) < target) {
        __nanosleep(ns);
        if (ns < 256) ns *= 2;
    }
}

CANS_D Task decode_ticket(const FusedArgs& a, unsigned t) {
    Task tk;
    if (t >= a.total) { tk.type = TASK_END; tk.k = tk.idx = tk.slot = 0; return tk; }
    const unsigned r = t / a.per_round;
    unsigned q = t - r * a.per_round;
    int s = 0;
    if (q >= a.slot_count[0]) {
        q -= a.slot_count[0];
        s = 1;
        if (a.nslots > 2 && q >= a.slot_count[1]) { q -= a.slot_count[1]; s = 2; }
    }
    tk.slot = s;
    tk.idx = (int)q;
    tk.k = (int)r - a.slot_off[s];
    tk.type = (tk.k >= 0 && tk.k < a.ax.nz) ? a.slot_type[s] : TASK_NONE;
    return tk;
}

// the (up to two) counters a task waits for; returns how many
CANS_D int task_deps(const FusedArgs& a, const Task& tk, const unsigned* (&c)[2], unsigned& target) {
    if (tk.type < 0 || tk.slot == 0) return 0;
    const unsigned* base = a.counters + (size_t)(tk.slot - 1) * a.cstride;
    target = a.slot_count[tk.slot - 1];
    c[0] = base + tk.k;
    if (tk.type == TASK_G && tk.k + 1 < a.ax.nz) { c[1] = base + tk.k + 1; return 2; }
    return 1;
}

// ---- streaming tasks: several items' loads are issued before the first use (memory-level parallelism) ----

// a7: gradient correction of rows [j0, j1) of plane k (eq. 2c; grad_pass.cuh)
template <int NT, int U>
CANS_D void grad_rows(const GradArgs& g, int k, int j0, int j1, int tid) {
    const size_t hx = (size_t)(g.nx >> 1);
    const size_t t0 = ((size_t)k * g.ny + j0) * hx;
    const size_t t1 = ((size_t)k * g.ny + j1) * hx;
    for (size_t base = t0 + tid; base < t1; base += (size_t)U * NT) {
        GradIn in[U];
#pragma unroll
        for (int q = 0; q < U; ++q)
            if (base + (size_t)q * NT < t1) in[q] = grad_load(g, base + (size_t)q * NT);
#pragma unroll
        for (int q = 0; q < U; ++q)
            if (base + (size_t)q * NT < t1) grad_apply(g, in[q]);
    }
}

extern __shared__ __align__(16) unsigned char cans_dyn_smem[];

template <int A, int B> struct MaxOf { static constexpr int value = A > B ? A : B; };

// shared-memory plan of one (PX, PY) pair; sizes in cplx (16 B) units: one FFT work buffer shared by the
// x and y tasks of the CTA, followed by both twiddle tables
template <class PX, class PY, int NFX, int TXC>
struct FusedSmem {
    static constexpr int WORK = MaxOf<NFX * PX::NPAD, PY::N * TXC>::value;
    static constexpr int TW = PX::TW_TOTAL + PY::TW_TOTAL;
    static constexpr size_t BYTES = sizeof(cplx) * (size_t)(WORK + TW);
};

// INV = false: pass A (X = [divergence +] forward x transform, Y = forward y transform)
// INV = true : pass C (Y = inverse y transform, X = inverse x transform, G = gradient rows)
template <class PX, class PY, int NFX, int TXC, int NT, bool INV>
__global__ void __launch_bounds__(NT, 2) fused_xy_kernel(const FusedArgs a) {
    typedef FusedSmem<PX, PY, NFX, TXC> L;
    typedef XPass<PX, NFX, NT, L::WORK> X;
    typedef YPass<PY, TXC, NT, L::WORK + PX::TW_TOTAL> Y;
    cplx* const sm = reinterpret_cast<cplx*>(cans_dyn_smem);
    __shared__ unsigned s_next;
    const int tid = threadIdx.x;
    const int nx = a.ax.nx, ny = a.ax.ny;
    const unsigned rowb = (unsigned)(nx * sizeof(double));

    // L2 prefetch of the HBM-resident input rows of a task (issued one task ahead of its loads)
    auto prefetch = [&](const Task& tk) {
        if (!INV && tk.type == TASK_X) {
            const int nr = 2 * NFX;
            const size_t ro = ((size_t)tk.k * ny + (size_t)nr * tk.idx) * (size_t)nx;
            if (a.mode) {
                if (tid < 3 * nr) {
                    const int fld = tid / nr, r = tid - fld * nr;
                    l2_prefetch_bulk((fld == 0 ? a.ax.u : (fld == 1 ? a.ax.v : a.ax.w)) + ro + (size_t)r * nx, rowb);
                }
            } else if (tid < nr) {
                l2_prefetch_bulk(a.ax.p + ro + (size_t)tid * nx, rowb);
            }
        } else if (INV && tk.type == TASK_Y) {
            // the y tiles of a plane together read the whole plane: each prefetches its share of rows
            const int nyt = (int)a.slot_count[tk.slot];
            const int j0 = (int)(((long)tk.idx * ny) / nyt);
            const int j1 = (int)(((long)(tk.idx + 1) * ny) / nyt);
            if (tid < j1 - j0) l2_prefetch_bulk(a.ay.p + ((size_t)tk.k * ny + j0 + tid) * (size_t)nx, rowb);
        } else if (INV && tk.type == TASK_G) {
            const int j0 = tk.idx * a.grows;
            const int nr = min(a.grows, ny - j0);
            if (tid < 3 * nr) {
                const int fld = tid / nr, r = tid - fld * nr;
                l2_prefetch_bulk((fld == 0 ? a.g.u : (fld == 1 ? a.g.v : a.g.w)) + ((size_t)tk.k * ny + j0 + r) * (size_t)nx, rowb);
            }
        }
    };

    X::load_twiddles(a.ax, sm, tid);
    Y::load_twiddles(a.ay, sm, tid);
    unsigned t2 = 0;                                     // thread 0: the ticket after next (already drawn)
    if (tid == 0) {
        s_next = atomicAdd(a.ticket, 1u);
        t2 = atomicAdd(a.ticket, 1u);
    }
    __syncthreads();
    Task cur = decode_ticket(a, s_next);
    __syncthreads();

    while (cur.type != TASK_END) {
        // thread 0 publishes the next ticket and draws the one after it (its latency hides behind this task),
        // then waits for the planes this task reads; the barrier publishes both to the CTA
        if (tid == 0) {
            s_next = t2;
            t2 = atomicAdd(a.ticket, 1u);
            const unsigned* c[2];
            unsigned target = 0;
            const int nd = task_deps(a, cur, c, target);
            for (int d = 0; d < nd; ++d) wait_counter(c[d], target);
            if (nd) __threadfence();
        }
        __syncthreads();
        const Task nxt = decode_ticket(a, s_next);
        prefetch(nxt);

        if (cur.type == TASK_X) {
            const long pair0 = (long)cur.k * (ny >> 1) + (long)cur.idx * NFX;
            const long lim = (long)(cur.k + 1) * (ny >> 1);
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
        } else if (cur.type == TASK_Y) {
            if (!INV) {
                Y::load_forward(a.ay, sm, cur.idx, cur.k, tid);
                __syncthreads();
                Y::pass1_fwd(sm, tid);
                __syncthreads();
                if (PY::R2 > 1) { Y::pass2_fwd(sm, tid); __syncthreads(); }
                Y::pass3_fwd(sm, tid);
                __syncthreads();
                Y::store_forward(a.ay, sm, cur.idx, cur.k, tid);
            } else {
                Y::load_inverse(a.ay, sm, cur.idx, cur.k, tid);
                __syncthreads();
                Y::pass3_inv(sm, tid);
                __syncthreads();
                if (PY::R2 > 1) { Y::pass2_inv(sm, tid); __syncthreads(); }
                Y::pass1_inv(sm, tid);
                __syncthreads();
                Y::store_inverse(a.ay, sm, cur.idx, cur.k, tid);
            }
        } else if (INV && cur.type == TASK_G) {
            const int j0 = cur.idx * a.grows;
            grad_rows<NT, 2>(a.g, cur.k, j0, min(j0 + a.grows, ny), tid);
        }

        __syncthreads();                                   // every thread's stores are issued ...
        if (tid == 0 && cur.type >= 0) {
            __threadfence();                               // ... and visible before the count moves
            atomicAdd(a.counters + (size_t)cur.slot * a.cstride + cur.k, 1u);
        }
        cur = nxt;
    }
}

template <class K>
static cudaError_t fused_set_smem(K kern, size_t bytes) {
    return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

// what: 0 = configure (sets *grid, *smem), 1 = launch pass A, 2 = launch pass C
template <class PX, class PY, int NFX, int TXC, int NT>
cudaError_t fused_run(int what, const FusedArgs* a, int num_sms, int* grid, size_t* smem, cudaStream_t st) {
    const size_t bytes = FusedSmem<PX, PY, NFX, TXC>::BYTES;
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
        *grid = occ * num_sms;                             // persistent: every CTA resident
        *smem = bytes;
        return cudaSuccess;
    }
    if (what == 1) ka<<<(unsigned)*grid, NT, *smem, st>>>(*a);
    else kc<<<(unsigned)*grid, NT, *smem, st>>>(*a);
    return cudaGetLastError();
}

// defined in cans_poisson.cu: routes to the per-nx translation units (fused_x*.cu)
bool fused_dispatch(int nx, int ny, int what, const FusedArgs* a, int num_sms, int* grid, size_t* smem,
                    cudaStream_t st, cudaError_t* err);
#endif

}  // namespace cans
