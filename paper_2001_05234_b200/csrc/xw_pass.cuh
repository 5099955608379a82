// xw_pass.cuh -- warp-per-line x transforms for the long lines (N = R1 * 32, R1 in {16, 24, 32}):
// the batched real-to-real transforms F^x of eq. 6 and their inverses, with the
// divergence of eq. 2b fused into the forward load.  Same mathematics, packing ("two real rows ->
// one complex line") and spectral slot layout as xy_pass.cuh; different machine mapping:
//
//   * ONE WARP owns a pair of rows from the first load to the last store: no CTA barrier anywhere, warps
//     drift apart freely, so one warp's loads overlap another warp's butterflies;
//   * 2-pass Cooley-Tukey in REGISTERS: lane p loads x[p + 32 m] (m < R1) straight from global memory --
//     2*R1 independent, perfectly coalesced 8-byte loads in flight per lane -- does the R1-point DFT over m,
//     applies W_N^(p k1), exchanges once through a padded per-warp shared-memory buffer, and lane k1 does
//     the 32-point DFT over p.  One shared-memory round trip instead of three;
//   * the spectrum is laid out in natural order in the same buffer for the real/imaginary separation
//     (post_forward / pre_inverse of xy_pass.cuh) and goes to global memory as coalesced 16-byte stores.
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
    template <bool DIV>
    static CANS_D void forward(const XYArgs& a, const cplx* __restrict__ tw, cplx* buf, size_t ro, int j, int k, int lane) {
        // phase 0: the two rows (or the divergence at them) in natural order -> buf[i] = (a_i, b_i), read from
        // global memory as coalesced 16-byte loads, UB column pairs per lane in flight at a time
        const size_t plane = (size_t)a.nx * a.ny;
        constexpr int NQ = H / 32;                       // column pairs per lane
        constexpr int UB = DIV ? 4 : (NQ < 16 ? NQ : 16);
        cplx v[R1];
        const bool direct = !DIV && a.kind == KIND_PP;   // periodic rows of a stored field: no staging needed
        if (direct) {
            // lane p takes x[p + 32 m] of both rows straight into registers: 2*R1 independent 8-byte loads,
            // every load instruction of the warp reads 256 contiguous bytes
#pragma unroll
            for (int m = 0; m < R1; ++m)
                v[m] = make_double2(__ldcg(a.p + ro + lane + 32 * m), __ldcg(a.p + ro + a.nx + lane + 32 * m));
        }
#pragma unroll 1
        for (int m0 = 0; m0 < (direct ? 0 : NQ); m0 += UB) {
            double2 fa[UB], fb[UB];
            if (!DIV) {
#pragma unroll
                for (int u = 0; u < UB; ++u) {
                    const int i0 = 2 * (lane + 32 * (m0 + u));
                    fa[u] = ld_p2(a.p + ro + i0);
                    fb[u] = ld_p2(a.p + ro + a.nx + i0);
                }
            } else {
                double2 ua[UB], ub[UB], v0[UB], v1[UB], v2[UB], wa[UB], wb[UB], wla[UB], wlb[UB];
                double ula0[UB], ulb0[UB];
                const double2 zero2 = make_double2(0.0, 0.0);
#pragma unroll
                for (int u = 0; u < UB; ++u) {
                    const int i0 = 2 * (lane + 32 * (m0 + u));
                    ua[u] = *reinterpret_cast<const double2*>(a.u + ro + i0);
                    ub[u] = *reinterpret_cast<const double2*>(a.u + ro + a.nx + i0);
                    // left neighbour of the pair: lane - 1 holds it, except for lane 0
                    ula0[u] = 0.0; ulb0[u] = 0.0;
                    if (lane == 0) {
                        if (i0 > 0) { ula0[u] = a.u[ro + i0 - 1]; ulb0[u] = a.u[ro + a.nx + i0 - 1]; }
                        else if (a.wrap_x) { ula0[u] = a.u[ro + a.nx - 1]; ulb0[u] = a.u[ro + 2 * (size_t)a.nx - 1]; }
                        else if (a.fx) { ula0[u] = a.fx[(size_t)k * a.ny + j]; ulb0[u] = a.fx[(size_t)k * a.ny + j + 1]; }
                    }
                    v1[u] = *reinterpret_cast<const double2*>(a.v + ro + i0);
                    v2[u] = *reinterpret_cast<const double2*>(a.v + ro + a.nx + i0);
                    if (j > 0) v0[u] = *reinterpret_cast<const double2*>(a.v + ro - a.nx + i0);
                    else if (a.wrap_y) v0[u] = *reinterpret_cast<const double2*>(a.v + ro + (size_t)(a.ny - 1) * a.nx + i0);
                    else if (a.fy) v0[u] = *reinterpret_cast<const double2*>(a.fy + (size_t)k * a.nx + i0);
                    else v0[u] = zero2;
                    wa[u] = *reinterpret_cast<const double2*>(a.w + ro + i0);
                    wb[u] = *reinterpret_cast<const double2*>(a.w + ro + a.nx + i0);
                    if (k > 0) {
                        wla[u] = *reinterpret_cast<const double2*>(a.w + ro - plane + i0);
                        wlb[u] = *reinterpret_cast<const double2*>(a.w + ro - plane + a.nx + i0);
                    } else if (a.wrap_z) {
                        wla[u] = *reinterpret_cast<const double2*>(a.w + ro + (size_t)(a.nz - 1) * plane + i0);
                        wlb[u] = *reinterpret_cast<const double2*>(a.w + ro + (size_t)(a.nz - 1) * plane + a.nx + i0);
                    } else if (a.fz) {
                        wla[u] = *reinterpret_cast<const double2*>(a.fz + (size_t)j * a.nx + i0);
                        wlb[u] = *reinterpret_cast<const double2*>(a.fz + (size_t)(j + 1) * a.nx + i0);
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
            }
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                const int i0 = 2 * (lane + 32 * (m0 + u));
                buf[i0] = make_double2(fa[u].x, fb[u].x);
                buf[i0 + 1] = make_double2(fa[u].y, fb[u].y);
            }
        }
        __syncwarp();
        if (!direct) {
#pragma unroll
            for (int m = 0; m < R1; ++m) {
                const int i = index_of_elem(lane + 32 * m, a.kind);
                v[m] = buf[i];
                if (kind_neg_odd(a.kind) && (i & 1)) v[m] = cneg(v[m]);
            }
            if (kind_mixed(a.kind)) {
#pragma unroll
                for (int m = 0; m < R1; ++m) v[m] = cmul(v[m], __ldg(a.wpre + lane + 32 * m));
            }
        }
        __syncwarp();                                   // natural-order rows fully read: reuse the buffer for the exchange
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
        __syncwarp();                                   // exchange buffer fully read: reuse it in natural order
        if (lane < R1) {
#pragma unroll
            for (int k2 = 0; k2 < 32; ++k2) buf[lane + R1 * k2] = w[k2];
        }
        __syncwarp();
#pragma unroll 4
        for (int s = lane; s < H; s += 32) {
            double2 oa, ob;
            if (kind_mixed(a.kind)) {
                post_forward(buf[s], buf[N - 1 - s], __ldg(a.wpost + s), a.kind, oa.x, oa.y, ob.x, ob.y);
            } else if (s == 0) {
                const cplx Z0 = buf[0], Zh = buf[H];
                const double c = (a.kind == KIND_PP) ? 1.0 : CANS_SQRT_HALF;
                oa = make_double2(Z0.x, c * Zh.x);
                ob = make_double2(Z0.y, c * Zh.y);
            } else {
                cplx wq = make_double2(1.0, 0.0);
                if (a.kind != KIND_PP) wq = __ldg(a.wpost + s);
                post_forward(buf[s], buf[N - s], wq, a.kind, oa.x, oa.y, ob.x, ob.y);
            }
            *reinterpret_cast<double2*>(a.p + ro + 2 * s) = oa;
            *reinterpret_cast<double2*>(a.p + ro + a.nx + 2 * s) = ob;
        }
        __syncwarp();                                   // buffer free for the warp's next pair
    }

    // ---- inverse: slots of rows (ro, ro + nx) -> the two real rows ----
    static CANS_D void inverse(const XYArgs& a, const cplx* __restrict__ tw, cplx* buf, size_t ro, int lane) {
        constexpr int NQ = H / 32;                       // slots per lane, all loaded before the first use
        {
            double2 ia[NQ], ib[NQ];
#pragma unroll
            for (int m = 0; m < NQ; ++m) {
                ia[m] = ld_p2(a.p + ro + 2 * (lane + 32 * m));
                ib[m] = ld_p2(a.p + ro + a.nx + 2 * (lane + 32 * m));
            }
#pragma unroll
            for (int m = 0; m < NQ; ++m) {
                const int s = lane + 32 * m;
                if (kind_mixed(a.kind)) {
                    cplx Zq, Zm;
                    pre_inverse(ia[m].x, ia[m].y, ib[m].x, ib[m].y, __ldg(a.wpost + s), a.kind, Zq, Zm);
                    buf[s] = Zq;
                    buf[N - 1 - s] = Zm;
                } else if (s == 0) {
                    const double c = (a.kind == KIND_PP) ? 1.0 : (1.0 / CANS_SQRT_HALF);
                    buf[0] = make_double2(ia[m].x, ib[m].x);
                    buf[H] = make_double2(c * ia[m].y, c * ib[m].y);
                } else {
                    cplx wq = make_double2(1.0, 0.0);
                    if (a.kind != KIND_PP) wq = __ldg(a.wpost + s);
                    cplx Zq, Zm;
                    pre_inverse(ia[m].x, ia[m].y, ib[m].x, ib[m].y, wq, a.kind, Zq, Zm);
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
        if (a.kind == KIND_PP) {
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
        __syncwarp();                                   // exchange buffer fully read: reuse it in natural order
        if (kind_mixed(a.kind)) {
#pragma unroll
            for (int m = 0; m < R1; ++m) v[m] = cmulc(v[m], __ldg(a.wpre + lane + 32 * m));
        }
#pragma unroll
        for (int m = 0; m < R1; ++m) {
            const int i = index_of_elem(lane + 32 * m, a.kind);
            buf[i] = (kind_neg_odd(a.kind) && (i & 1)) ? cneg(v[m]) : v[m];
        }
        __syncwarp();
#pragma unroll
        for (int m = 0; m < NQ; ++m) {
            const int i0 = 2 * (lane + 32 * m);
            const cplx z0 = buf[i0], z1 = buf[i0 + 1];
            *reinterpret_cast<double2*>(a.p + ro + i0) = make_double2(z0.x, z1.x);
            *reinterpret_cast<double2*>(a.p + ro + a.nx + i0) = make_double2(z0.y, z1.y);
        }
        __syncwarp();
    }
#endif
};

}  // namespace cans
