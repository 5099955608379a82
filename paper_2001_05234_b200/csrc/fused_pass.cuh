// fused_pass.cuh -- passes A and C of the projection as persistent task kernels fused through L2.
//
//   pass A = a1 + a2 + a3 : divergence (eq. 2b) -> forward x transform -> forward y transform
//   pass C = a5 + a6 + a7 : inverse y -> inverse x (eq. 6) -> u -= dt G Phi (eq. 2c)
//
// A k-plane (C5: 6.3 MB) does not fit one SM's shared memory but fits the 126 MB L2 many times, so the
// intermediate planes of a pass never have to reach HBM.  One persistent CTA per SM draws TICKETS from a
// global counter.  Tickets are ordered in ROUNDS; round r holds, in this order, the tasks of up to three
// SLOTS, slot s working on plane k = r - off[s]:
//     pass A (projection):  D(r)  divergence rows     X(r-1)  x transforms     Y(r-2)  y transforms
//     pass A (Poisson):     X(r)                      Y(r-1)
//     pass C:               Y(r)  inverse y           X(r-1)  inverse x        G(r-3)  gradient rows
// A task of slot s waits until every task of slot s-1 on its plane has signalled (G also waits for the
// plane above, whose Phi it reads).  A task therefore only ever waits for tasks with SMALLER tickets,
// which are finished or held by a running CTA: no deadlock, no co-residency requirement.
//
// Latency hiding: the input of the NEXT transform task is copied global -> shared (cp.async.cg, no
// register staging, L2-coherent) into a staging buffer while the CURRENT task computes in the work
// buffer; divergence / gradient tasks stream through registers with several pairs of loads in flight
// and have their HBM rows prefetched into L2 (cp.async.bulk.prefetch.L2) one task ahead.
#pragma once
#include <cuda_runtime.h>
#include "xy_pass.cuh"
#include "grad_pass.cuh"

namespace cans {

enum TaskType : int { TASK_END = -2, TASK_NONE = -1, TASK_X = 0, TASK_Y = 1, TASK_G = 2, TASK_D = 3 };

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
    int drows, grows;           // rows per divergence / gradient task
};

struct Task { int type, k, idx, slot; };

// tiling of the fused kernels per transform length (host and device agree through these)
constexpr int FUSED_NT = 512;
constexpr int FUSED_DROWS = 8;
constexpr int FUSED_GROWS = 8;
constexpr int fused_nfx(int nx) { return nx >= 768 ? 4 : 8; }       // row pairs per x task
constexpr int fused_txc(int ny) { return ny <= 768 ? 8 : 4; }       // complex columns per y task
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
CANS_D unsigned ld_relaxed_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}
CANS_D void l2_prefetch_bulk(const void* p, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;\n" ::"l"(p), "r"(bytes) : "memory");
}
CANS_D void fx_cp_async16(void* smem_dst, const void* gmem_src) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem_src) : "memory");
}
CANS_D void fx_cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
CANS_D void fx_cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }

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

// a1: divergence of rows [j0, j1) of plane k -> p (eq. 2b; same arithmetic as XPass::load_forward<true>)
template <int NT, int U>
CANS_D void div_rows(const XYArgs& a, int k, int j0, int j1, int tid) {
    const int hx = a.nx >> 1;
    const int nitems = (j1 - j0) * hx;
    const size_t plane = (size_t)a.nx * a.ny;
    const double rz = a.rdzf[k];
    const double2 zero2 = make_double2(0.0, 0.0);
    for (int base = tid; base < nitems; base += U * NT) {
        double2 ua[U], v1[U], v0[U], wa[U], wl[U];
        double ul[U];
        size_t off[U];
#pragma unroll
        for (int q = 0; q < U; ++q) {
            const int it = base + q * NT;
            if (it < nitems) {
                const int r = it / hx;
                const int i0 = 2 * (it - r * hx);
                const int j = j0 + r;
                const size_t o = (size_t)k * plane + (size_t)j * a.nx + i0;
                off[q] = o;
                ua[q] = *reinterpret_cast<const double2*>(a.u + o);
                ul[q] = (i0 > 0) ? a.u[o - 1] : (a.wrap_x ? a.u[o + a.nx - 1] : 0.0);
                v1[q] = *reinterpret_cast<const double2*>(a.v + o);
                v0[q] = (j > 0) ? *reinterpret_cast<const double2*>(a.v + o - a.nx)
                                : (a.wrap_y ? *reinterpret_cast<const double2*>(a.v + o + (size_t)(a.ny - 1) * a.nx) : zero2);
                wa[q] = *reinterpret_cast<const double2*>(a.w + o);
                wl[q] = (k > 0) ? *reinterpret_cast<const double2*>(a.w + o - plane)
                                : (a.wrap_z ? *reinterpret_cast<const double2*>(a.w + o + (size_t)(a.nz - 1) * plane) : zero2);
            }
        }
#pragma unroll
        for (int q = 0; q < U; ++q) {
            const int it = base + q * NT;
            if (it < nitems) {
                double2 f;
                f.x = div_value(ua[q].x - ul[q], v1[q].x - v0[q].x, wa[q].x - wl[q].x, a.rdx, a.rdy, rz, a.rdt);
                f.y = div_value(ua[q].y - ua[q].x, v1[q].y - v0[q].y, wa[q].y - wl[q].y, a.rdx, a.rdy, rz, a.rdt);
                *reinterpret_cast<double2*>(a.p + off[q]) = f;
            }
        }
    }
}

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

// shared-memory plan of one (PX, PY) pair; sizes in cplx (16 B) units
template <class PX, class PY, int NFX, int TXC>
struct FusedSmem {
    static constexpr int WORK = MaxOf<NFX * PX::NPAD, PY::N * TXC>::value;     // FFT work buffer
    static constexpr int TW = PX::TW_TOTAL + PY::TW_TOTAL;                     // both twiddle tables
    static constexpr int STAGE = MaxOf<NFX * PX::N, PY::N * TXC>::value;       // raw input of the next task
    static constexpr size_t BYTES = sizeof(cplx) * (size_t)(WORK + TW + STAGE);
};


// INV = false: pass A (D = divergence rows, X = forward x transform, Y = forward y transform)
// INV = true : pass C (Y = inverse y transform, X = inverse x transform, G = gradient rows)
template <class PX, class PY, int NFX, int TXC, int NT, bool INV>
__global__ void __launch_bounds__(NT, 1) fused_xy_kernel(const FusedArgs a) {
    typedef FusedSmem<PX, PY, NFX, TXC> L;
    typedef XPass<PX, NFX, NT, L::WORK> X;
    typedef YPass<PY, TXC, NT, L::WORK + PX::TW_TOTAL> Y;
    cplx* sm = reinterpret_cast<cplx*>(cans_dyn_smem);
    double* S = reinterpret_cast<double*>(sm + L::WORK + L::TW);
    __shared__ unsigned s_next;
    __shared__ int s_ready;
    const int tid = threadIdx.x;
    const int nx = a.ax.nx, ny = a.ax.ny;

    // copy the raw input of a transform task into the staging buffer (asynchronously), or prefetch the
    // HBM rows of a streaming task into L2.  Requires the task's dependencies to be satisfied.
    auto stage_in = [&](const Task& tk) {
        if (tk.type == TASK_X) {
            const double* src = a.ax.p + ((size_t)tk.k * ny + (size_t)2 * NFX * tk.idx) * (size_t)nx;
            for (int c = tid; c < NFX * PX::N; c += NT) fx_cp_async16(S + 2 * c, src + 2 * c);
        } else if (tk.type == TASK_Y) {
            const double* src = a.ay.p + (size_t)tk.k * ny * (size_t)nx + 2 * (size_t)tk.idx * TXC;
            for (int c = tid; c < PY::N * TXC; c += NT) {
                const int j = c / TXC;
                const int q = c - j * TXC;
                fx_cp_async16(S + 2 * c, src + (size_t)j * nx + 2 * q);
            }
        } else if (tk.type == TASK_D || tk.type == TASK_G) {
            const int rows = (tk.type == TASK_D) ? a.drows : a.grows;
            const int j0 = tk.idx * rows;
            const int nr = min(rows, ny - j0);
            if (tid < 3 * nr) {
                const int fld = tid / nr, r = tid - fld * nr;
                const double* u = (tk.type == TASK_D) ? a.ax.u : a.g.u;
                const double* v = (tk.type == TASK_D) ? a.ax.v : a.g.v;
                const double* w = (tk.type == TASK_D) ? a.ax.w : a.g.w;
                const double* src = (fld == 0 ? u : (fld == 1 ? v : w)) + ((size_t)tk.k * ny + j0 + r) * (size_t)nx;
                l2_prefetch_bulk(src, (unsigned)(nx * sizeof(double)));
            }
        }
        fx_cp_async_commit();
    };
    auto block_wait = [&](const Task& tk) {
        if (tid == 0) {
            const unsigned* c[2];
            unsigned target = 0;
            const int nd = task_deps(a, tk, c, target);
            for (int d = 0; d < nd; ++d) wait_counter(c[d], target);
            if (nd) __threadfence();
        }
        __syncthreads();
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
    if (cur.type == TASK_END) return;
    block_wait(cur);                                     // (also orders the read of s_next before its rewrite)
    stage_in(cur);

    while (true) {
        // thread 0 publishes the next ticket, draws the one after it (latency hidden behind this task)
        // and probes the next task's dependencies; the answers are used after the unpack
        unsigned c0 = 0, c1 = 0, target = 0;
        int nd = 0;
        if (tid == 0) {
            const unsigned tn = t2;
            s_next = tn;
            t2 = atomicAdd(a.ticket, 1u);
            const Task nt = decode_ticket(a, tn);
            const unsigned* c[2];
            nd = task_deps(a, nt, c, target);
            if (nd > 0) c0 = ld_relaxed_u32(c[0]);
            if (nd > 1) c1 = ld_relaxed_u32(c[1]);
        }
        // the staged input of the current transform task has landed: unpack it into the work buffer
        if (cur.type == TASK_X || cur.type == TASK_Y) {
            fx_cp_async_wait_all();
            __syncthreads();
            if (cur.type == TASK_X) {
                if (!INV) X::unpack_forward(a.ax, sm, S, tid); else X::unpack_inverse(a.ax, sm, S, tid);
            } else {
                if (!INV) Y::unpack_forward(a.ay, sm, S, tid); else Y::unpack_inverse(a.ay, sm, S, tid);
            }
        }
        if (tid == 0) {
            const int ready = (nd < 1 || c0 >= target) && (nd < 2 || c1 >= target);
            if (ready && nd) __threadfence();             // relaxed load + fence = acquire
            s_ready = ready;
        }
        __syncthreads();                                   // staging buffer free, work buffer filled
        const Task nxt = decode_ticket(a, s_next);
        const bool ready = s_ready != 0;
        if (ready) stage_in(nxt);                          // overlaps the whole computation below

        if (cur.type == TASK_X) {
            const long pair0 = (long)cur.k * (ny >> 1) + (long)cur.idx * NFX;
            const long lim = (long)(cur.k + 1) * (ny >> 1);
            if (!INV) {
                X::pass1_fwd(sm, tid);
                __syncthreads();
                if (PX::R2 > 1) { X::pass2_fwd(sm, tid); __syncthreads(); }
                X::pass3_fwd(sm, tid);
                __syncthreads();
                X::store_forward(a.ax, sm, pair0, lim, tid);
            } else {
                X::pass3_inv(sm, tid);
                __syncthreads();
                if (PX::R2 > 1) { X::pass2_inv(sm, tid); __syncthreads(); }
                X::pass1_inv(sm, tid);
                __syncthreads();
                X::store_inverse(a.ax, sm, pair0, lim, tid);
            }
        } else if (cur.type == TASK_Y) {
            if (!INV) {
                Y::pass1_fwd(sm, tid);
                __syncthreads();
                if (PY::R2 > 1) { Y::pass2_fwd(sm, tid); __syncthreads(); }
                Y::pass3_fwd(sm, tid);
                __syncthreads();
                Y::store_forward(a.ay, sm, cur.idx, cur.k, tid);
            } else {
                Y::pass3_inv(sm, tid);
                __syncthreads();
                if (PY::R2 > 1) { Y::pass2_inv(sm, tid); __syncthreads(); }
                Y::pass1_inv(sm, tid);
                __syncthreads();
                Y::store_inverse(a.ay, sm, cur.idx, cur.k, tid);
            }
        } else if (!INV && cur.type == TASK_D) {
            const int j0 = cur.idx * a.drows;
            div_rows<NT, 2>(a.ax, cur.k, j0, min(j0 + a.drows, ny), tid);
        } else if (INV && cur.type == TASK_G) {
            const int j0 = cur.idx * a.grows;
            grad_rows<NT, 2>(a.g, cur.k, j0, min(j0 + a.grows, ny), tid);
        }

        __syncthreads();                                   // every thread's stores are issued ...
        if (tid == 0 && cur.type >= 0) {
            __threadfence();                               // ... and visible before the count moves
            atomicAdd(a.counters + (size_t)cur.slot * a.cstride + cur.k, 1u);
        }
        if (nxt.type == TASK_END) break;
        if (!ready) {
            block_wait(nxt);
            stage_in(nxt);
        }
        cur = nxt;
    }
    fx_cp_async_wait_all();
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
        if (oa < 1 || oc < 1) return cudaErrorLaunchOutOfResources;
        *grid = num_sms;                                   // one persistent CTA per SM
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
