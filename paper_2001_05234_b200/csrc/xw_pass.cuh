// xw_pass.cuh -- warp-per-line x transforms for the long lines (N = R1 * 32, R1 in {16, 24, 32}):
// the batched real-to-real transforms F^x of eq. 6 and their inverses, with the
// divergence of eq. 2b fused into the forward load.  Same mathematics, packing ("two real rows ->
// one complex line") and spectral slot layout as xy_pass.cuh; different machine mapping:
//
//   * ONE WARP owns a pair of rows from the first load to the last store: no CTA barrier anywhere, warps
//     drift apart freely, so one warp's loads overlap another warp's butterflies;
//   * 2-pass Cooley-Tukey in REGISTERS: lane p holds the FFT input elements p + 32 m (m < R1) -- periodic rows as
//     2*R1 coalesced 8-byte loads straight from global memory, non-periodic rows as 16-byte sample pairs whose odd
//     sample goes to the mirrored lane by one shuffle (Makhoul's permutation is a lane mirror), the fused divergence
//     through one staging pass in the warp's buffer -- does the R1-point DFT over m, applies W_N^(p k1), exchanges once
//     through a padded per-warp shared-memory buffer, and lane k1 does the 32-point DFT over p.  One shared-memory
//     round trip instead of three;
//   * the spectrum is laid out in natural order in the same buffer for the real/imaginary separation
//     (post_forward / pre_inverse of xy_pass.cuh) and goes to global memory as coalesced 16-byte stores;
//   * one kernel per class of boundary pair (KC: PP; NN / DD; ND / DN), so the periodic kernels carry no twiddle code.
//
// Forward:  X[k1 + R1 k2] = sum_p W_32^(p k2) * W_N^(p k1) * sum_m W_R1^(m k1) x[p + 32 m]
// Inverse:  the same factorisation run backwards with conjugated roots (unnormalised).
#pragma once
#include "xy_pass.cuh"

namespace cans {

// cos(2 pi m / D) for the extra composite radices (quarter-wave symmetric tables)
template <> CANS_HD double tab_cos<32>(int m) {
    m = ((m % 32) + 32) % 32;
    if (m > 16) m = 32 - m;
    const bool neg = m > 8;
    if (neg) m = 16 - m;
    double c;
    switch (m) {
        case 0: c = 1.0; break;
        case 1: c = 0.98078528040323044913; break;
        case 2: c = 0.92387953251128675613; break;
        case 3: c = 0.83146961230254523708; break;
        case 4: c = 0.70710678118654752440; break;
        case 5: c = 0.55557023301960222474; break;
        case 6: c = 0.38268343236508977173; break;
        case 7: c = 0.19509032201612826785; break;
        default: c = 0.0; break;
    }
    return neg ? -c : c;
}
template <> CANS_HD double tab_cos<24>(int m) {
    m = ((m % 24) + 24) % 24;
    if (m > 12) m = 24 - m;
    const bool neg = m > 6;
    if (neg) m = 12 - m;
    double c;
    switch (m) {
        case 0: c = 1.0; break;
        case 1: c = 0.96592582628906828675; break;
        case 2: c = 0.86602540378443864676; break;
        case 3: c = 0.70710678118654752440; break;
        case 4: c = 0.5; break;
        case 5: c = 0.25881904510252076235; break;
        default: c = 0.0; break;
    }
    return neg ? -c : c;
}
template <bool INV> struct Dft<32, INV> { static CANS_HD void run(cplx (&v)[32]) { DftComposite<4, 8, 32, INV>::run(v); } };
template <bool INV> struct Dft<24, INV> { static CANS_HD void run(cplx (&v)[24]) { DftComposite<3, 8, 24, INV>::run(v); } };

constexpr int XW_WARPS = 4;                      // warps (row pairs) per CTA
inline bool xw_supported(int n) { return n == 512 || n == 768 || n == 1024; }

template <int N_, int R1_>
struct XWPass {
    static constexpr int N = N_, R1 = R1_, H = N_ / 2;
    static_assert(R1_ * 32 == N_, "N = R1 * 32");
    static constexpr int XSTRIDE = 33;                               // padded row of the exchange buffer
    static constexpr int BUF = (R1 * XSTRIDE > N) ? R1 * XSTRIDE : N;   // cplx per warp

    // FFT input element e -> natural index along the line (Makhoul's even/odd permutation for NN / DD)
    static CANS_HD int index_of_elem(int e, int kind) {
        if (kind == KIND_PP) return e;
        return (e < H) ? 2 * e : 2 * (N - 1 - e) + 1;
    }
    // Staging position of natural sample i of a periodic line: lane L stores the pair (2e, 2e+1), a stride of two 16-byte
    // units that would fold the eight lanes of a quarter warp onto four bank groups; flipping the low bit in every
    // second group of eight makes the pair stores and the unit-stride reads both conflict free.
    static CANS_HD int stage_pos(int i) { return i ^ ((i >> 3) & 1); }

#if defined(__CUDACC__)
    // W_N^(lane k1), k1 = 1..R1-1, applied to v (conjugated for the inverse): every 8th root is read from the
    // plan's table (exact), the ones between are products with W_N^lane (at most 7 roundings) -- 4 table
    // reads per lane instead of R1 - 1 keep the L1 data pipe for the exchange
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

    // ---- forward: rows (ro, ro + nx) of the field (or the divergence at those rows) -> slots ----
    // KC: class of the boundary pair (0 = PP, 1 = NN / DD, 2 = ND / DN), a compile-time switch so that the periodic kernels
    // carry none of the permutation / twiddle code; the pair inside a class is the run-time a.kind
    template <bool DIV, int KC>
    static CANS_D void forward(const XYArgs& a, const cplx* __restrict__ tw, cplx* buf, size_t ro, int j, int k, int lane) {
        constexpr bool pp = KC == 0, mixed = KC == 2;
        const int kind = pp ? (int)KIND_PP : a.kind;
        // phase 0: the FFT input elements lane + 32 m of the packed line (row a) + i (row b) in registers.
        //   * stored periodic rows: 8-byte loads straight from global memory (every load instruction of the warp reads
        //     256 contiguous bytes), no staging;
        //   * stored non-periodic rows: 16-byte loads of the sample pairs (2e, 2e+1), e = lane + 32 m; Makhoul's
        //     permutation sends sample 2e to element e (this lane) and sample 2e+1 to element N-1-e = (31 - lane) +
        //     32 (R1-1-m), i.e. to the mirrored lane: one shuffle, no staging;
        //   * fused divergence: computed pair by pair in batches and staged once in the warp's buffer at the
        //     element's position (periodic: an XOR swizzle makes the pair stores conflict free).
        const size_t plane = (size_t)a.nx * a.ny;
        constexpr int NQ = H / 32;                       // column pairs per lane
        constexpr int UB = 4;
        cplx v[R1];
        if (!DIV && pp) {
#pragma unroll
            for (int m = 0; m < R1; ++m)
                v[m] = make_double2(__ldcg(a.p + ro + lane + 32 * m), __ldcg(a.p + ro + a.nx + lane + 32 * m));
        } else if (!DIV) {
            double2 fa[NQ], fb[NQ];
#pragma unroll
            for (int m = 0; m < NQ; ++m) {
                fa[m] = ld_p2(a.p + ro + 2 * (lane + 32 * m));
                fb[m] = ld_p2(a.p + ro + a.nx + 2 * (lane + 32 * m));
            }
            const double sgn = kind_neg_odd(kind) ? -1.0 : 1.0;
#pragma unroll
            for (int m = 0; m < NQ; ++m) {
                v[m] = make_double2(fa[m].x, fb[m].x);
                v[R1 - 1 - m] = make_double2(__shfl_xor_sync(0xffffffffu, sgn * fa[m].y, 31),
                                             __shfl_xor_sync(0xffffffffu, sgn * fb[m].y, 31));
            }
        } else {
#pragma unroll 1
            for (int m0 = 0; m0 < NQ; m0 += UB) {
                double2 fa[UB], fb[UB];
                double2 ua[UB], ub[UB], v0[UB], v1[UB], v2[UB], wa[UB], wb[UB], wla[UB], wlb[UB];
                double ula0[UB], ulb0[UB];
                const double2 zero2 = make_double2(0.0, 0.0);
#pragma unroll
                for (int u = 0; u < UB; ++u) {
                    const int i0 = 2 * (lane + 32 * (m0 + u));
                    ua[u] = ldg_stream2(a.u + ro + i0);
                    ub[u] = ldg_stream2(a.u + ro + a.nx + i0);
                    // left neighbour of the pair: lane - 1 holds it, except for lane 0
                    ula0[u] = 0.0; ulb0[u] = 0.0;
                    if (lane == 0) {
                        if (i0 > 0) { ula0[u] = a.u[ro + i0 - 1]; ulb0[u] = a.u[ro + a.nx + i0 - 1]; }
                        else if (a.wrap_x) { ula0[u] = a.u[ro + a.nx - 1]; ulb0[u] = a.u[ro + 2 * (size_t)a.nx - 1]; }
                        else if (a.fx) { ula0[u] = a.fx[(size_t)k * a.ny + j]; ulb0[u] = a.fx[(size_t)k * a.ny + j + 1]; }
                    }
                    v1[u] = ldg_stream2(a.v + ro + i0);
                    v2[u] = ldg_stream2(a.v + ro + a.nx + i0);
                    if (j > 0) v0[u] = ldg_stream2(a.v + ro - a.nx + i0);
                    else if (a.wrap_y) v0[u] = ldg_stream2(a.v + ro + (size_t)(a.ny - 1) * a.nx + i0);
                    else if (a.fy) v0[u] = ldg_stream2(a.fy + (size_t)k * a.nx + i0);
                    else v0[u] = zero2;
                    wa[u] = ldg_stream2(a.w + ro + i0);
                    wb[u] = ldg_stream2(a.w + ro + a.nx + i0);
                    if (k > 0) {
                        wla[u] = ldg_stream2(a.w + ro - plane + i0);
                        wlb[u] = ldg_stream2(a.w + ro - plane + a.nx + i0);
                    } else if (a.wrap_z) {
                        wla[u] = ldg_stream2(a.w + ro + (size_t)(a.nz - 1) * plane + i0);
                        wlb[u] = ldg_stream2(a.w + ro + (size_t)(a.nz - 1) * plane + a.nx + i0);
                    } else if (a.fz) {
                        wla[u] = ldg_stream2(a.fz + (size_t)j * a.nx + i0);
                        wlb[u] = ldg_stream2(a.fz + (size_t)(j + 1) * a.nx + i0);
                    } else { wla[u] = zero2; wlb[u] = zero2; }
                }
                const double rz = a.rdzf[k];
#pragma unroll
                for (int u = 0; u < UB; ++u) {
                    const double pa = __shfl_up_sync(0xffffffffu, ua[u].y, 1);
                    const double pb = __shfl_up_sync(0xffffffffu, ub[u].y, 1);
                    const double ula = (lane == 0) ? ula0[u] : pa;
                    const double ulb = (lane == 0) ? ulb0[u] : pb;
                    fa[u].x = div_value(ua[u].x - ula, v1[u].x - v0[u].x, wa[u].x - wla[u].x, a.rdx, a.rdy, rz, a.rdt);
                    fa[u].y = div_value(ua[u].y - ua[u].x, v1[u].y - v0[u].y, wa[u].y - wla[u].y, a.rdx, a.rdy, rz, a.rdt);
                    fb[u].x = div_value(ub[u].x - ulb, v2[u].x - v1[u].x, wb[u].x - wlb[u].x, a.rdx, a.rdy, rz, a.rdt);
                    fb[u].y = div_value(ub[u].y - ub[u].x, v2[u].y - v1[u].y, wb[u].y - wlb[u].y, a.rdx, a.rdy, rz, a.rdt);
                }
#pragma unroll
                for (int u = 0; u < UB; ++u) {
                    const int e = lane + 32 * (m0 + u);          // samples 2e, 2e+1
                    const cplx z0 = make_double2(fa[u].x, fb[u].x);
                    cplx z1 = make_double2(fa[u].y, fb[u].y);
                    if (pp) {
                        buf[stage_pos(2 * e)] = z0;
                        buf[stage_pos(2 * e + 1)] = z1;
                    } else {
                        if (kind_neg_odd(kind)) z1 = cneg(z1);
                        buf[e] = z0;
                        buf[N - 1 - e] = z1;
                    }
                }
            }
            __syncwarp();
#pragma unroll
            for (int m = 0; m < R1; ++m) v[m] = buf[pp ? stage_pos(lane + 32 * m) : lane + 32 * m];
            __syncwarp();                               // staged elements fully read: reuse the buffer for the exchange
        }
        if (mixed) {
            const cplx wl = __ldg(a.wpre + lane);
#pragma unroll
            for (int m = 0; m < R1; ++m) v[m] = cmul(v[m], cmul(wl, a.wstep[m]));
        }
        Dft<R1, false>::run(v);
        apply_twiddles<false>(v, tw, lane);
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) buf[k1 * XSTRIDE + lane] = v[k1];
        __syncwarp();
        cplx w[32];
        if (lane < R1) {
#pragma unroll
            for (int p = 0; p < 32; ++p) w[p] = buf[lane * XSTRIDE + p];
            Dft<32, false>::run(w);
        }
        // quarter-wave post-twiddles of this lane's slots: all loads issued here, behind the exchange below
        cplx wq[NQ];
        if (!pp) {
#pragma unroll
            for (int m = 0; m < NQ; ++m) wq[m] = __ldg(a.wpost + lane + 32 * m);
        }
        __syncwarp();                                   // exchange buffer fully read: reuse it in natural order
        if (lane < R1) {
#pragma unroll
            for (int k2 = 0; k2 < 32; ++k2) buf[lane + R1 * k2] = w[k2];
        }
        __syncwarp();
#pragma unroll
        for (int m = 0; m < NQ; ++m) {
            const int s = lane + 32 * m;
            double2 oa, ob;
            if (mixed) {
                post_forward(buf[s], buf[N - 1 - s], wq[m], kind, oa.x, oa.y, ob.x, ob.y);
            } else if (s == 0) {
                const cplx Z0 = buf[0], Zh = buf[H];
                const double c = pp ? 1.0 : CANS_SQRT_HALF;
                oa = make_double2(Z0.x, c * Zh.x);
                ob = make_double2(Z0.y, c * Zh.y);
            } else {
                post_forward(buf[s], buf[N - s], pp ? make_double2(1.0, 0.0) : wq[m], kind, oa.x, oa.y, ob.x, ob.y);
            }
            *reinterpret_cast<double2*>(a.p + ro + 2 * s) = oa;
            *reinterpret_cast<double2*>(a.p + ro + a.nx + 2 * s) = ob;
        }
        __syncwarp();                                   // buffer free for the warp's next pair
    }

    // ---- inverse: slots of rows (ro, ro + nx) -> the two real rows ----
    template <int KC>
    static CANS_D void inverse(const XYArgs& a, const cplx* __restrict__ tw, cplx* buf, size_t ro, int lane) {
        constexpr bool pp = KC == 0, mixed = KC == 2;
        const int kind = pp ? (int)KIND_PP : a.kind;
        constexpr int NQ = H / 32;                       // slots per lane, all loaded before the first use
        {
            double2 ia[NQ], ib[NQ];
            cplx wq[NQ];
#pragma unroll
            for (int m = 0; m < NQ; ++m) {
                ia[m] = ld_p2(a.p + ro + 2 * (lane + 32 * m));
                ib[m] = ld_p2(a.p + ro + a.nx + 2 * (lane + 32 * m));
            }
            if (!pp) {
#pragma unroll
                for (int m = 0; m < NQ; ++m) wq[m] = __ldg(a.wpost + lane + 32 * m);
            }
#pragma unroll
            for (int m = 0; m < NQ; ++m) {
                const int s = lane + 32 * m;
                if (mixed) {
                    cplx Zq, Zm;
                    pre_inverse(ia[m].x, ia[m].y, ib[m].x, ib[m].y, wq[m], kind, Zq, Zm);
                    buf[s] = Zq;
                    buf[N - 1 - s] = Zm;
                } else if (s == 0) {
                    const double c = pp ? 1.0 : (1.0 / CANS_SQRT_HALF);
                    buf[0] = make_double2(ia[m].x, ib[m].x);
                    buf[H] = make_double2(c * ia[m].y, c * ib[m].y);
                } else {
                    cplx Zq, Zm;
                    pre_inverse(ia[m].x, ia[m].y, ib[m].x, ib[m].y, pp ? make_double2(1.0, 0.0) : wq[m], kind, Zq, Zm);
                    buf[s] = Zq;
                    buf[N - s] = Zm;
                }
            }
        }
        __syncwarp();
        cplx w[32];
        if (lane < R1) {
#pragma unroll
            for (int k2 = 0; k2 < 32; ++k2) w[k2] = buf[lane + R1 * k2];
            Dft<32, true>::run(w);
        }
        __syncwarp();                                   // natural-order buffer fully read: reuse as exchange buffer
        if (lane < R1) {
#pragma unroll
            for (int p = 0; p < 32; ++p) buf[lane * XSTRIDE + p] = w[p];
        }
        __syncwarp();
        cplx v[R1];
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) v[k1] = buf[k1 * XSTRIDE + lane];
        apply_twiddles<true>(v, tw, lane);
        Dft<R1, true>::run(v);
        if (pp) {
            // periodic lines need no permutation: lane p holds x[p + 32 m], so every store instruction of the
            // warp writes 256 contiguous bytes of a row straight from registers
#pragma unroll
            for (int m = 0; m < R1; ++m) {
                a.p[ro + lane + 32 * m] = v[m].x;
                a.p[ro + a.nx + lane + 32 * m] = v[m].y;
            }
            __syncwarp();
            return;
        }
        // Non-periodic lines: element e = lane + 32 m is sample 2e (m < R1/2); sample 2e+1 is element N-1-e, held by
        // the mirrored lane as its v[R1-1-m]: one shuffle, then the pair goes out as a coalesced 16-byte store.
        if (mixed) {
            const cplx wl = __ldg(a.wpre + lane);
#pragma unroll
            for (int m = 0; m < R1; ++m) v[m] = cmulc(v[m], cmul(wl, a.wstep[m]));
        }
        const double sgn = kind_neg_odd(kind) ? -1.0 : 1.0;
#pragma unroll
        for (int m = 0; m < NQ; ++m) {
            const double z1x = sgn * __shfl_xor_sync(0xffffffffu, v[R1 - 1 - m].x, 31);
            const double z1y = sgn * __shfl_xor_sync(0xffffffffu, v[R1 - 1 - m].y, 31);
            const int i0 = 2 * (lane + 32 * m);
            *reinterpret_cast<double2*>(a.p + ro + i0) = make_double2(v[m].x, z1x);
            *reinterpret_cast<double2*>(a.p + ro + a.nx + i0) = make_double2(v[m].y, z1y);
        }
        __syncwarp();
    }
#endif
};

}  // namespace cans
