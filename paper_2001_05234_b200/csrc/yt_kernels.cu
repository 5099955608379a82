// yt_kernels.cu -- persistent TMA-fed y transform kernels (yt_pass.cuh) and their launcher.
#include "yt_kernels.cuh"

namespace cans {

extern __shared__ __align__(1024) unsigned char cans_dyn_smem_1k[];

template <int N, int R1, bool INV, int KC>
__global__ void __launch_bounds__(YT_NT, 1) yt_kernel(const XYArgs a, const cplx* __restrict__ tw,
                                                      const __grid_constant__ CUtensorMap tmap, int ntx, long ntiles) {
    typedef YTPass<N, R1, KC> W;
    cplx* bufs = reinterpret_cast<cplx*>(cans_dyn_smem_1k);
    __shared__ __align__(8) unsigned long long s_bar[2];
    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        mbar_init(&s_bar[0], 1);
        mbar_init(&s_bar[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    // tile t = (plane k, column tile c): boxes of 16 doubles x 256 rows at (16 c, k N + 256 box)
    // FIRST: all boxes at once.  Otherwise box by box, each as soon as the write-back of the same box of the tile
    // that occupied this buffer (one bulk group per box, oldest first) has finished reading shared memory.
    // boxes [box0, box1) of tile t into buffer bsel; the first box of a tile arms the buffer's mbarrier for the whole tile
    auto issue_load = [&](long t, int bsel, bool first, int box0, int box1) {
        const int kl = (int)(t / ntx);
        const int c = (int)(t - (long)kl * ntx);
        const int k = a.k0 + kl;
        if (box0 == 0) mbar_expect_tx(&s_bar[bsel], W::TILE_BYTES);
#pragma unroll
        for (int box = 0; box < W::NBOX; ++box) {
            if (box < box0 || box >= box1) continue;
            if (!first) {
                // box b may be refilled once the write-back group of box b has read it: at most NBOX-1-b younger groups pending
                if (box == 0) tma_store_wait_read_pending<W::NBOX - 1>();
                else if (box == 1) tma_store_wait_read_pending<(W::NBOX > 2 ? W::NBOX - 2 : 0)>();
                else if (box == 2) tma_store_wait_read_pending<(W::NBOX > 3 ? W::NBOX - 3 : 0)>();
                else tma_store_wait_read_pending<0>();
            }
            tma_load_2d(bufs + (size_t)bsel * W::TILE + (size_t)box * YT_BOX_ROWS * YT_COLS, &tmap, 2 * YT_COLS * c,
                        k * N + box * YT_BOX_ROWS, &s_bar[bsel]);
        }
    };
    long t = blockIdx.x;
    if (t >= ntiles) return;
    if (tid == 0) issue_load(t, 0, true, 0, W::NBOX);
    unsigned phases = 0u;
    int b = 0;
    // NBUF = 2: the copy of the next tile into the other buffer is issued before this tile is transformed.  NBUF = 1 (one
    // tile fills the shared memory: N = 1024): the next tile is copied into the same buffer box by box, each box as soon
    // as its write-back has read it -- the transform of a tile overlaps nothing but the tail of the previous write-back.
    constexpr int NBUF = W::NBUF;
    for (; t < ntiles; t += gridDim.x) {
        const long tn = t + gridDim.x;
        // The thread that issued the write-back of the previous tile (same buffer b^1) must wait for each box to be read
        // before refilling it: it asks for the first box now (its write-back group is the oldest) and for the others
        // between its own two transform phases, when they have drained -- it hardly ever blocks, so its warp does not
        // keep the other seven waiting at the tile barrier.
        if (NBUF == 2 && tid == 0 && tn < ntiles) issue_load(tn, b ^ 1, false, 0, 1);
        mbar_wait(&s_bar[b], (phases >> b) & 1u);
        phases ^= 1u << b;
        cplx* T = bufs + (size_t)b * W::TILE;
        if (INV) {
            W::slots_in(a, T, warp, lane);
            if (NBUF == 2 && tid == 0 && tn < ntiles) issue_load(tn, b ^ 1, false, 1, W::NBOX);
            W::column_inverse(a, T, warp, tw, lane);
        } else {
            W::column_forward(a, T, warp, tw, lane, [&]() {
                if (NBUF == 2 && tid == 0 && tn < ntiles) issue_load(tn, b ^ 1, false, 1, W::NBOX);
            });
            W::slots_out(a, T, warp, lane);
        }
        fence_proxy_async_smem();               // this thread's shared-memory writes -> visible to the TMA unit
        __syncthreads();
        if (tid == 0) {
            const int kl = (int)(t / ntx);
            const int c = (int)(t - (long)kl * ntx);
            const int k = a.k0 + kl;
            for (int box = 0; box < W::NBOX; ++box)
            {
                tma_store_2d(&tmap, 2 * YT_COLS * c, k * N + box * YT_BOX_ROWS, T + (size_t)box * YT_BOX_ROWS * YT_COLS);
                tma_store_commit();             // one bulk group per box
            }
            if (NBUF == 1 && tn < ntiles) issue_load(tn, 0, false, 0, W::NBOX);
        }
        if (NBUF == 2) b ^= 1;
    }
    if (tid == 0) tma_store_wait_all();
}

template <int N, int R1, int KC>
static cudaError_t yt_launch_k(int op, const XYArgs& a, const cplx* tw, const CUtensorMap* tmap, int max_ctas, cudaStream_t st) {
    const size_t smem = YTPass<N, R1, KC>::NBUF * sizeof(cplx) * (size_t)YTPass<N, R1, KC>::TILE;
    if (op == OP_CONFIGURE) {
        cudaError_t e = cudaFuncSetAttribute(yt_kernel<N, R1, false, KC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(yt_kernel<N, R1, true, KC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        return e;
    }
    const int ntx = a.nx / 2 / YT_COLS;
    const long ntiles = (long)ntx * a.nk;
    const unsigned grid = (unsigned)(ntiles < max_ctas ? ntiles : max_ctas);
    if (op == OP_Y_FWD) yt_kernel<N, R1, false, KC><<<grid, YT_NT, smem, st>>>(a, tw, *tmap, ntx, ntiles);
    else yt_kernel<N, R1, true, KC><<<grid, YT_NT, smem, st>>>(a, tw, *tmap, ntx, ntiles);
    return cudaGetLastError();
}

// one kernel per class of boundary pair (yt_kind_class): the periodic kernels carry no permutation / twiddle code
template <int N, int R1>
static cudaError_t yt_launch_n(int op, const XYArgs& a, const cplx* tw, const CUtensorMap* tmap, int max_ctas, cudaStream_t st) {
    if (op == OP_CONFIGURE) {                            // plan time: every class (the opt-in is per kernel)
        cudaError_t e = yt_launch_k<N, R1, 0>(op, a, tw, tmap, max_ctas, st);
        if (e == cudaSuccess) e = yt_launch_k<N, R1, 1>(op, a, tw, tmap, max_ctas, st);
        if (e == cudaSuccess) e = yt_launch_k<N, R1, 2>(op, a, tw, tmap, max_ctas, st);
        return e;
    }
    switch (yt_kind_class(a.kind)) {
        case 0: return yt_launch_k<N, R1, 0>(op, a, tw, tmap, max_ctas, st);
        case 1: return yt_launch_k<N, R1, 1>(op, a, tw, tmap, max_ctas, st);
        default: return yt_launch_k<N, R1, 2>(op, a, tw, tmap, max_ctas, st);
    }
}

// the field as a 2-D tensor: nx doubles per row, ny*nz rows; boxes of 16 doubles x 256 rows, 128-byte swizzle
cudaError_t yt_make_tensor_map(CUtensorMap* tmap, const double* p, int nx, int ny, int nz) {
    return make_tensor_map_2d(tmap, p, (unsigned long long)nx, (unsigned long long)ny * nz,
                              (unsigned long long)nx * sizeof(double), 2 * YT_COLS, YT_BOX_ROWS, CU_TENSOR_MAP_SWIZZLE_128B);
}

bool yt_launch(int n, int op, const XYArgs& a, const cplx* tw, const CUtensorMap* tmap, int max_ctas, cudaStream_t st,
               cudaError_t* err) {
    switch (n) {
        case 512: *err = yt_launch_n<512, 16>(op, a, tw, tmap, max_ctas, st); return true;
        case 768: *err = yt_launch_n<768, 24>(op, a, tw, tmap, max_ctas, st); return true;
        case 1024: *err = yt_launch_n<1024, 32>(op, a, tw, tmap, max_ctas, st); return true;
        default: return false;
    }
}

}  // namespace cans
