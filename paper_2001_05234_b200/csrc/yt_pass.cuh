// yt_pass.cuh -- TMA-fed y transforms (N = R1 * 32: 512, 768 with two tile buffers, 1024 with one): F^y of eq. 6
// and its inverse.  Mathematics and slot layout as YPass (xy_pass.cuh).
//
// A persistent CTA of 8 warps (one per SM) walks over tiles of 8 complex columns x N rows:
//   * the TMA unit copies the tile global -> shared (cp.async.bulk.tensor.2d, boxes of 16 doubles x 256 rows,
//     SWIZZLE_128B, completion on an mbarrier) and, after the transform, shared -> global -- no thread issues a
//     global load or store, and the copy of tile n+1 / the write-back of tile n-1 overlap the transform of tile n
//     (two buffers);
//   * warp f owns column f of the tile from the first to the last shared-memory access: the 2-pass register FFT (as
//     xw_pass.cuh; the permutation of the non-periodic pairs is folded into its first load / last store) and the
//     real/imaginary separation all happen in place with __syncwarp only; one CTA barrier per tile hands the
//     finished tile to the TMA store;
//   * one kernel per class of boundary pair (KC), as in xw_pass.cuh.
// With the 128-byte swizzle, element (row e, column f) sits at complex index e*8 + (f ^ (e & 7)): the eight lanes of a
// quarter warp reading one column at eight consecutive (or XOR-permuted) rows hit eight different 16-byte bank
// groups, so every column access of the FFT is conflict free without padding.
#pragma once
#include "xw_pass.cuh"
#include "tma_util.cuh"

namespace cans {

constexpr int YT_COLS = 8;                       // complex columns per tile = warps per CTA
constexpr int YT_NT = YT_COLS * 32;
constexpr int YT_BOX_ROWS = 256;
inline bool yt_supported(int n) { return n == 512 || n == 768 || n == 1024; }

// KC: class of the boundary pair, a compile-time switch so that the periodic kernels carry none of the registers of the
// permutation / twiddle paths: 0 = PP, 1 = NN / DD, 2 = ND / DN (the pair inside a class is the run-time `kind`)
constexpr int yt_kind_class(int kind) { return kind == KIND_PP ? 0 : (kind >= KIND_ND ? 2 : 1); }

template <int N_, int R1_, int KC>
struct YTPass {
    static constexpr int N = N_, R1 = R1_, H = N_ / 2;
    static constexpr bool IS_PP = KC == 0, IS_MIXED = KC == 2;
    static_assert(R1_ * 32 == N_ && N_ % YT_BOX_ROWS == 0, "N = R1 * 32, whole TMA boxes");
    static constexpr int TILE = N * YT_COLS;                         // cplx per buffer
    static constexpr int NBOX = N / YT_BOX_ROWS;
    static constexpr unsigned TILE_BYTES = (unsigned)(TILE * sizeof(cplx));
    static constexpr int NBUF = (2 * TILE_BYTES <= 200 * 1024) ? 2 : 1;      // tile buffers that fit the shared memory

#if defined(__CUDACC__)
    static CANS_D int at(int e, int f) { return e * YT_COLS + (f ^ (e & 7)); }

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

    // Row of the tile holding FFT input element e (Makhoul's even/odd permutation for every non-periodic pair; the
    // identity for PP): e < H -> row 2e, e >= H -> row 2(N-1-e)+1.
    static CANS_D int row_of_elem(int e, int kind) {
        if (IS_PP) return e;
        return (e < H) ? 2 * e : 2 * (N - 1 - e) + 1;
    }
    // Lane p owns the FFT input elements p + 32 m.  For the non-periodic pairs elements m and m + R1/2 sit in an even and an
    // odd row; lanes with bit 2 set touch the odd row first, so that the eight rows of one shared-memory access differ
    // modulo 8 (conflict free under the swizzle) -- the permutation costs no pass of its own.
    static CANS_D void load_elems(const XYArgs& a, const cplx* t, int f, int lane, cplx (&v)[R1]) {
        const int kind = a.kind;
        if (IS_PP) {
#pragma unroll
            for (int m = 0; m < R1; ++m) v[m] = t[at(lane + 32 * m, f)];
            return;
        }
        const bool odd_first = (lane & 4) != 0;
#pragma unroll
        for (int m = 0; m < R1 / 2; ++m) {
            const int je = 2 * (lane + 32 * m);                           // element m
            const int jo = 2 * (N - 1 - (lane + 32 * (m + R1 / 2))) + 1;   // element m + R1/2
            const cplx x0 = t[at(odd_first ? jo : je, f)];
            const cplx x1 = t[at(odd_first ? je : jo, f)];
            v[m] = odd_first ? x1 : x0;
            const cplx zo = odd_first ? x0 : x1;
            v[m + R1 / 2] = kind_neg_odd(kind) ? cneg(zo) : zo;
        }
        if (IS_MIXED) {
            const cplx wl = __ldg(a.wpre + lane);
#pragma unroll
            for (int m = 0; m < R1; ++m) v[m] = cmul(v[m], cmul(wl, a.wstep[m]));
        }
    }
    static CANS_D void store_elems(const XYArgs& a, cplx* t, int f, int lane, cplx (&v)[R1]) {
        const int kind = a.kind;
        if (IS_PP) {
#pragma unroll
            for (int m = 0; m < R1; ++m) t[at(lane + 32 * m, f)] = v[m];
            return;
        }
        if (IS_MIXED) {
            const cplx wl = __ldg(a.wpre + lane);
#pragma unroll
            for (int m = 0; m < R1; ++m) v[m] = cmulc(v[m], cmul(wl, a.wstep[m]));
        }
        const bool odd_first = (lane & 4) != 0;
#pragma unroll
        for (int m = 0; m < R1 / 2; ++m) {
            const int je = 2 * (lane + 32 * m);
            const int jo = 2 * (N - 1 - (lane + 32 * (m + R1 / 2))) + 1;
            const cplx ze = v[m];
            const cplx zo = kind_neg_odd(kind) ? cneg(v[m + R1 / 2]) : v[m + R1 / 2];
            t[at(odd_first ? jo : je, f)] = odd_first ? zo : ze;
            t[at(odd_first ? je : jo, f)] = odd_first ? ze : zo;
        }
    }

    // rows as loaded (natural order) -> natural-order spectrum, in place in column f (unnormalised)
    // `mid` runs between the two passes (the kernel's elected thread issues TMA work there)
    template <class Mid>
    static CANS_D void column_forward(const XYArgs& a, cplx* t, int f, const cplx* __restrict__ tw, int lane, Mid&& mid) {
        cplx v[R1];
        load_elems(a, t, f, lane, v);
        Dft<R1, false>::run(v);
        apply_twiddles<false>(v, tw, lane);
        __syncwarp();
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) t[at(k1 * 32 + (lane ^ k1), f)] = v[k1];
        mid();
        __syncwarp();
        cplx w[32];
        if (lane < R1) {
#pragma unroll
            for (int p = 0; p < 32; ++p) w[p] = t[at(lane * 32 + (p ^ lane), f)];
            Dft<32, false>::run(w);
        }
        __syncwarp();
        if (lane < R1) {
#pragma unroll
            for (int k2 = 0; k2 < 32; ++k2) t[at(lane + R1 * k2, f)] = w[k2];
        }
        __syncwarp();
    }
    static CANS_D void column_inverse(const XYArgs& a, cplx* t, int f, const cplx* __restrict__ tw, int lane) {
        cplx w[32];
        if (lane < R1) {
#pragma unroll
            for (int k2 = 0; k2 < 32; ++k2) w[k2] = t[at(lane + R1 * k2, f)];
            Dft<32, true>::run(w);
        }
        __syncwarp();
        if (lane < R1) {
#pragma unroll
            for (int p = 0; p < 32; ++p) t[at(lane * 32 + (p ^ lane), f)] = w[p];
        }
        __syncwarp();
        cplx v[R1];
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) v[k1] = t[at(k1 * 32 + (lane ^ k1), f)];
        apply_twiddles<true>(v, tw, lane);
        Dft<R1, true>::run(v);
        __syncwarp();
        store_elems(a, t, f, lane, v);       // FFT output elements -> rows (the inverse of load_elems)
        __syncwarp();
    }

    // natural-order spectrum -> slot rows (2s, 2s+1), in place through registers (YPass::store_forward)
    static CANS_D void slots_out(const XYArgs& a, cplx* t, int f, int lane) {
        constexpr int NS = H / 32;
        cplx zq[NS], zm[NS], wq[NS];
        if (!IS_PP) {                         // post-twiddles: issued before the shared-memory reads
#pragma unroll
            for (int m = 0; m < NS; ++m) wq[m] = __ldg(a.wpost + lane + 32 * m);
        }
#pragma unroll
        for (int m = 0; m < NS; ++m) {
            const int s = lane + 32 * m;
            zq[m] = t[at(s, f)];
            zm[m] = t[at(IS_MIXED ? N - 1 - s : (s == 0 ? H : N - s), f)];
        }
        __syncwarp();
#pragma unroll
        for (int m = 0; m < NS; ++m) {
            const int s = lane + 32 * m;
            cplx r0, r1;
            if (s == 0 && !IS_MIXED) {
                const double c = IS_PP ? 1.0 : CANS_SQRT_HALF;
                r0 = make_double2(zq[m].x, zq[m].y);
                r1 = make_double2(c * zm[m].x, c * zm[m].y);
            } else {
                double A0, A1, B0, B1;
                post_forward(zq[m], zm[m], IS_PP ? make_double2(1.0, 0.0) : wq[m], IS_PP ? (int)KIND_PP : a.kind, A0, A1, B0, B1);
                r0 = make_double2(A0, B0);
                r1 = make_double2(A1, B1);
            }
            // rows 2s and 2s+1: lanes 0-3 of every group of eight write the even row first and lanes 4-7 the odd
            // one, so that the eight rows of one store instruction differ modulo 8 (conflict free under the swizzle)
            const bool odd_first = (lane & 4) != 0;
            t[at(2 * s + (odd_first ? 1 : 0), f)] = odd_first ? r1 : r0;
            t[at(2 * s + (odd_first ? 0 : 1), f)] = odd_first ? r0 : r1;
        }
        __syncwarp();
    }
    // slot rows -> natural-order spectrum, in place through registers (YPass::load_inverse)
    static CANS_D void slots_in(const XYArgs& a, cplx* t, int f, int lane) {
        constexpr int NS = H / 32;
        cplx r0[NS], r1[NS], wq[NS];
        if (!IS_PP) {
#pragma unroll
            for (int m = 0; m < NS; ++m) wq[m] = __ldg(a.wpost + lane + 32 * m);
        }
#pragma unroll
        for (int m = 0; m < NS; ++m) {
            const int s = lane + 32 * m;
            const bool odd_first = (lane & 4) != 0;        // as in slots_out: eight different rows modulo 8 per load
            const cplx x0 = t[at(2 * s + (odd_first ? 1 : 0), f)];
            const cplx x1 = t[at(2 * s + (odd_first ? 0 : 1), f)];
            r0[m] = odd_first ? x1 : x0;
            r1[m] = odd_first ? x0 : x1;
        }
        __syncwarp();
#pragma unroll
        for (int m = 0; m < NS; ++m) {
            const int s = lane + 32 * m;
            if (s == 0 && !IS_MIXED) {
                const double c = IS_PP ? 1.0 : (1.0 / CANS_SQRT_HALF);
                t[at(0, f)] = make_double2(r0[m].x, r0[m].y);
                t[at(H, f)] = make_double2(c * r1[m].x, c * r1[m].y);
            } else {
                cplx Zq, Zm;
                pre_inverse(r0[m].x, r1[m].x, r0[m].y, r1[m].y, IS_PP ? make_double2(1.0, 0.0) : wq[m], IS_PP ? (int)KIND_PP : a.kind, Zq, Zm);
                t[at(s, f)] = Zq;
                t[at(IS_MIXED ? N - 1 - s : N - s, f)] = Zm;
            }
        }
        __syncwarp();
    }
#endif
};

}  // namespace cans
