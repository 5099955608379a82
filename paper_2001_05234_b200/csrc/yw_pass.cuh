// yw_pass.cuh -- y transforms for the long lines (N = R1 * 32, R1 in {16, 24, 32}) with a warp per column:
// F^y of eq. 6 and its inverse along the strided direction.  Mathematics, packing
// (two adjacent real columns = one complex column) and slot layout are those of YPass (xy_pass.cuh).
//
// A CTA of YW_WARPS warps owns a tile of YW_TXC complex columns x N rows of one k-plane:
//   1. all threads copy the tile global -> shared with every 16-byte load issued before the first use
//      (rows of 16*YW_TXC contiguous bytes; the input permutation / pre-processing is applied on the way);
//   2. a warp transforms its columns one after the other, each IN PLACE in the tile with the 2-pass register FFT of xw_pass.cuh (lane p
//      takes rows p + 32 m, R1-point DFTs, twiddle, one exchange through the column's own rows with an XOR
//      swizzle, 32-point DFTs) -- only __syncwarp inside;
//   3. all threads post-process and write the tile back as coalesced rows.
// Two CTA barriers per tile instead of five, one shared-memory exchange instead of three.
// Rows are padded to YW_TXC + 1 complex numbers so that a lane-per-row access of one column is conflict free.
#pragma once
#include "xw_pass.cuh"

namespace cans {

constexpr int YW_TXC = 8;                        // complex columns per CTA: rows of 128 contiguous bytes
constexpr int YW_WARPS = 4;                      // warps per CTA, each transforms YW_TXC / YW_WARPS columns in turn
constexpr int YW_NT = YW_WARPS * 32;
constexpr int YW_ROWS = YW_NT / YW_TXC;          // rows covered by one cooperative pass of the CTA
inline bool yw_supported(int n) { return n == 512 || n == 768 || n == 1024; }

template <int N_, int R1_>
struct YWPass {
    static constexpr int N = N_, R1 = R1_, H = N_ / 2;
    static_assert(R1_ * 32 == N_, "N = R1 * 32");
    static constexpr int RS = YW_TXC + 1;                            // padded row stride (cplx)
    static constexpr int TILE = N * RS;                              // cplx per CTA

#if defined(__CUDACC__)
    // base = element (row 0, real column 2*c0) of plane k
    static CANS_D double* tile_base(const XYArgs& a, int ctile, int k) {
        return a.p + (size_t)k * a.nx * a.ny + 2 * (size_t)ctile * YW_TXC;
    }

    // W_N^(lane k1), k1 = 1..R1-1, applied to v (conjugated for the inverse).  Two CTAs' tiles leave almost no
    // L1, so only every 8th root is read from the plan's table (exact); the ones between are products with
    // W_N^lane -- at most 7 roundings, far inside the 1e-11 parity bar.
    template <bool INV>
    static CANS_D void apply_twiddles(cplx (&v)[R1], const cplx* __restrict__ tw, int lane) {
        cplx anchor[R1 / 8];
#pragma unroll
        for (int g = 0; g < R1 / 8; ++g) anchor[g] = __ldg(tw + (g == 0 ? 1 : 8 * g) * 32 + lane);
        const cplx w1 = anchor[0];
        cplx wk = w1;
#pragma unroll
        for (int k1 = 1; k1 < R1; ++k1) {
            if ((k1 & 7) == 0) wk = anchor[k1 / 8];
            else if (k1 > 1) wk = cmul(wk, w1);
            v[k1] = INV ? cmulc(v[k1], wk) : cmul(v[k1], wk);
        }
    }

    // ---- in-place column transforms (one warp; col = &tile[f], element e at col[e * RS]) ----
    // natural-order input, natural-order output, unnormalised; exchange rows k1*32 + (p ^ k1)
    static CANS_D void column_forward(cplx* col, const cplx* __restrict__ tw, int lane) {
        cplx v[R1];
#pragma unroll
        for (int m = 0; m < R1; ++m) v[m] = col[(lane + 32 * m) * RS];
        Dft<R1, false>::run(v);
        apply_twiddles<false>(v, tw, lane);
        __syncwarp();                                   // every lane has read its rows
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) col[(k1 * 32 + (lane ^ k1)) * RS] = v[k1];
        __syncwarp();
        cplx w[32];
        if (lane < R1) {
#pragma unroll
            for (int p = 0; p < 32; ++p) w[p] = col[(lane * 32 + (p ^ lane)) * RS];
            Dft<32, false>::run(w);
        }
        __syncwarp();
        if (lane < R1) {
#pragma unroll
            for (int k2 = 0; k2 < 32; ++k2) col[(lane + R1 * k2) * RS] = w[k2];
        }
    }
    static CANS_D void column_inverse(cplx* col, const cplx* __restrict__ tw, int lane) {
        cplx w[32];
        if (lane < R1) {
#pragma unroll
            for (int k2 = 0; k2 < 32; ++k2) w[k2] = col[(lane + R1 * k2) * RS];
            Dft<32, true>::run(w);
        }
        __syncwarp();
        if (lane < R1) {
#pragma unroll
            for (int p = 0; p < 32; ++p) col[(lane * 32 + (p ^ lane)) * RS] = w[p];
        }
        __syncwarp();
        cplx v[R1];
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) v[k1] = col[(k1 * 32 + (lane ^ k1)) * RS];
        apply_twiddles<true>(v, tw, lane);
        Dft<R1, true>::run(v);
        __syncwarp();
#pragma unroll
        for (int m = 0; m < R1; ++m) col[(lane + 32 * m) * RS] = v[m];
    }

    // ---- cooperative tile phases (all YW_NT threads) ----
    // rows j -> FFT input element e (Makhoul permutation, DD sign), as YPass::load_forward
    static CANS_D void load_forward(const XYArgs& a, cplx* tile, int ctile, int k, int tid) {
        const double* base = tile_base(a, ctile, k);
        constexpr int ITERS = N / YW_ROWS;              // rows per thread
        constexpr int UB = ITERS / 4;                   // four batches of 8..16 independent 16-byte loads
        static_assert(ITERS % UB == 0, "batches must tile the rows");
        const int f = tid % YW_TXC;
        const int j0 = tid / YW_TXC;
#pragma unroll 1
        for (int it0 = 0; it0 < ITERS; it0 += UB) {
            cplx z[UB];
#pragma unroll
            for (int u = 0; u < UB; ++u) z[u] = ld_p2(base + (size_t)(j0 + YW_ROWS * (it0 + u)) * a.nx + 2 * f);
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                const int j = j0 + YW_ROWS * (it0 + u);
                const int e = elem_of_index<N>(j, a.kind);
                cplx zz = (kind_neg_odd(a.kind) && (j & 1)) ? cneg(z[u]) : z[u];
                if (kind_mixed(a.kind)) zz = cmul(zz, __ldg(a.wpre + e));
                tile[e * RS + f] = zz;
            }
        }
    }
    // natural-order spectrum -> slots (rows 2s, 2s+1), as YPass::store_forward with identity frequency map
    static CANS_D void store_forward(const XYArgs& a, const cplx* tile, int ctile, int k, int tid) {
        double* base = tile_base(a, ctile, k);
        const int f = tid % YW_TXC;
#pragma unroll 4
        for (int s = tid / YW_TXC; s < H; s += YW_ROWS) {
            double2 r0, r1;
            if (kind_mixed(a.kind)) {
                double A0, A1, B0, B1;
                post_forward(tile[s * RS + f], tile[(N - 1 - s) * RS + f], __ldg(a.wpost + s), a.kind, A0, A1, B0, B1);
                r0 = make_double2(A0, B0);
                r1 = make_double2(A1, B1);
            } else if (s == 0) {
                const cplx Z0 = tile[f], Zh = tile[H * RS + f];
                const double c = (a.kind == KIND_PP) ? 1.0 : CANS_SQRT_HALF;
                r0 = make_double2(Z0.x, Z0.y);
                r1 = make_double2(c * Zh.x, c * Zh.y);
            } else {
                cplx wq = make_double2(1.0, 0.0);
                if (a.kind != KIND_PP) wq = __ldg(a.wpost + s);
                double A0, A1, B0, B1;
                post_forward(tile[s * RS + f], tile[(N - s) * RS + f], wq, a.kind, A0, A1, B0, B1);
                r0 = make_double2(A0, B0);
                r1 = make_double2(A1, B1);
            }
            *reinterpret_cast<double2*>(base + (size_t)(2 * s) * a.nx + 2 * f) = r0;
            *reinterpret_cast<double2*>(base + (size_t)(2 * s + 1) * a.nx + 2 * f) = r1;
        }
    }
    // slots -> natural-order spectrum, as YPass::load_inverse
    static CANS_D void load_inverse(const XYArgs& a, cplx* tile, int ctile, int k, int tid) {
        const double* base = tile_base(a, ctile, k);
        constexpr int ITERS = H / YW_ROWS;              // slots per thread
        constexpr int UB = ITERS / 4;                   // four batches of 2 x (4..8) independent 16-byte loads
        static_assert(ITERS % UB == 0, "batches must tile the slots");
        const int f = tid % YW_TXC;
        const int s0 = tid / YW_TXC;
#pragma unroll 1
        for (int it0 = 0; it0 < ITERS; it0 += UB) {
            double2 r0[UB], r1[UB];
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                const int s = s0 + YW_ROWS * (it0 + u);
                r0[u] = ld_p2(base + (size_t)(2 * s) * a.nx + 2 * f);
                r1[u] = ld_p2(base + (size_t)(2 * s + 1) * a.nx + 2 * f);
            }
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                const int s = s0 + YW_ROWS * (it0 + u);
                if (kind_mixed(a.kind)) {
                    cplx Zq, Zm;
                    pre_inverse(r0[u].x, r1[u].x, r0[u].y, r1[u].y, __ldg(a.wpost + s), a.kind, Zq, Zm);
                    tile[s * RS + f] = Zq;
                    tile[(N - 1 - s) * RS + f] = Zm;
                } else if (s == 0) {
                    const double c = (a.kind == KIND_PP) ? 1.0 : (1.0 / CANS_SQRT_HALF);
                    tile[f] = make_double2(r0[u].x, r0[u].y);
                    tile[H * RS + f] = make_double2(c * r1[u].x, c * r1[u].y);
                } else {
                    cplx wq = make_double2(1.0, 0.0);
                    if (a.kind != KIND_PP) wq = __ldg(a.wpost + s);
                    cplx Zq, Zm;
                    pre_inverse(r0[u].x, r1[u].x, r0[u].y, r1[u].y, wq, a.kind, Zq, Zm);
                    tile[s * RS + f] = Zq;
                    tile[(N - s) * RS + f] = Zm;
                }
            }
        }
    }
    // element e -> row j, as YPass::store_inverse
    static CANS_D void store_inverse(const XYArgs& a, const cplx* tile, int ctile, int k, int tid) {
        double* base = tile_base(a, ctile, k);
        const int f = tid % YW_TXC;
#pragma unroll 4
        for (int j = tid / YW_TXC; j < N; j += YW_ROWS) {
            const int e = elem_of_index<N>(j, a.kind);
            cplx z = tile[e * RS + f];
            if (kind_mixed(a.kind)) z = cmulc(z, __ldg(a.wpre + e));
            if (kind_neg_odd(a.kind) && (j & 1)) z = cneg(z);
            *reinterpret_cast<double2*>(base + (size_t)j * a.nx + 2 * f) = z;
        }
    }
#endif
};

}  // namespace cans
