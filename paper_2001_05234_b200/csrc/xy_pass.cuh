// xy_pass.cuh -- phase functions of the batched real-to-real transforms along x and y
// (F^x, F^y of eq. 6; DFT for periodic, DCT-II/III for Neumann-Neumann, DST-II/III for
// Dirichlet-Dirichlet pairs), with the divergence of eq. 2b fused into the first load.
//
// Method ("two-for-one"): two REAL lines a, b are transformed by ONE complex FFT of z = a + i b.
//   PP   : Z = FFT(z);  A_q = (Z_q + conj Z_{n-q})/2,  B_q = (Z_q - conj Z_{n-q})/(2i)
//   NN   : v_j = x_{2j}, v_{n-1-j} = x_{2j+1} (Makhoul's permutation, P:L222 ref [21]);
//          C_q = Re(w^q V_q), C_{n-q} = -Im(w^q V_q), w = exp(-i pi/(2n))
//   DD   : x_j -> (-1)^j x_j, then as NN; the slot of C'_q holds sine mode n-1-q.
//   ND/DN: (mixed pairs, DCT-IV / DST-IV) the same permutation (ND also negates the odd samples), a
//          pre-twiddle v_m -> v_m exp(-i pi m / n), V = FFT(v): V_{n-1-q} = conj V_q for a real line, and with
//          G_q = exp(-i pi (2q+1)/(4n)) V_q the coefficients are (Re G_q, -Im G_q) = cosine modes (q, n-1-q) for ND,
//          sine modes (n-1-q, q) for DN.  The inverse runs the same steps backwards (conjugated).
// Spectral ("slot") layout of a line of n reals: positions (2s, 2s+1), s = 1..n/2-1, hold
// (Re A_s, Im A_s) for PP or (C_s, C_{n-s}) for NN/DD; positions (0, 1) hold modes (0, n/2).  Mixed pairs: positions
// (2s, 2s+1), s = 0..n/2-1, hold (Re G_s, -Im G_s).
// The eigenvalue of every position is tabulated by the plan (plan_tables.hpp), so the layout is private.
//
// x pass: the pair is two adjacent rows (j, j+1) of a plane; line index runs along x (contiguous).
// y pass: the pair is two adjacent columns (i, i+1), i.e. one double2 per row; line index runs along y.
//
// Every phase is a function of (tid, block coordinates); phases are separated by block barriers in
// xy_kernels.cuh.  No value is carried in registers across phases.
#pragma once
#include "fft_core.cuh"

namespace cans {

// Geometry + tables shared by the x/y kernels (passed by value as a kernel parameter).
struct XYArgs {
    int nx, ny, nz;
    int k0, nk;             // planes [k0, k0 + nk) handled by this launch (a batch of consecutive k-planes)
    int kind;               // Kind of THIS direction
    const cplx* tw;         // pass twiddles, FftPlan::TW_TOTAL entries
    const cplx* wpost;      // NN / DD: exp(-i pi q / (2n)); ND / DN: exp(-i pi (2q+1) / (4n)); q = 0..n/2-1
    const cplx* wpre;       // ND / DN only: exp(-i pi m / n), m = 0..n-1
    cplx wstep[32];         // ND / DN, warp-level kernels (n = 32 R1): wstep[m] = wpre[32 m] -- the pre-twiddle of element
                            // lane + 32 m is wpre[lane] * wstep[m]: one table load per lane, the steps come from the
                            // kernel's parameter bank (uniform reads, no memory latency at the end of the transform)
    double* p;              // field transformed in place
    // fused divergence (x forward only): f = (du*rdx + dv*rdy + dw*rdzf[k]) * rdt
    const double* u;
    const double* v;
    const double* w;
    const double* rdzf;     // 1/dzf[k]
    double rdx, rdy, rdt;
    int wrap_x, wrap_y, wrap_z;   // 1 if that direction is periodic (lower face = wrapped value), else 0
    // boundary-normal velocity on the lower face of a non-periodic direction (cans_projection_set_lower_face), or
    // NULL (=> 0, no penetration): fx[j + ny*k], fy[i + nx*k], fz[i + nx*j]
    const double* fx;
    const double* fy;
    const double* fz;
};

// natural index i of a line  ->  FFT input element (and whether the sample is negated)
template <int N>
CANS_HD int elem_of_index(int i, int kind) {
    if (kind == KIND_PP) return i;
    return (i & 1) ? (N - 1 - (i >> 1)) : (i >> 1);
}

// (Z_q, Z_{n-q}) -> the four reals stored at slot q of lines a and b
CANS_HD void post_forward(cplx Zq, cplx Zm, cplx wq, int kind, double& A0, double& A1, double& B0, double& B1) {
    cplx A = make_double2(0.5 * (Zq.x + Zm.x), 0.5 * (Zq.y - Zm.y));
    cplx B = make_double2(0.5 * (Zq.y + Zm.y), 0.5 * (Zm.x - Zq.x));
    if (kind != KIND_PP) {
        A = cmul(A, wq);
        B = cmul(B, wq);
        A.y = -A.y;
        B.y = -B.y;
    }
    A0 = A.x; A1 = A.y; B0 = B.x; B1 = B.y;
}

// inverse of post_forward
CANS_HD void pre_inverse(double A0, double A1, double B0, double B1, cplx wq, int kind, cplx& Zq, cplx& Zm) {
    cplx A = make_double2(A0, A1), B = make_double2(B0, B1);
    if (kind != KIND_PP) {
        A = cmulc(make_double2(A0, -A1), wq);
        B = cmulc(make_double2(B0, -B1), wq);
    }
    Zq = make_double2(A.x - B.y, A.y + B.x);
    Zm = make_double2(A.x + B.y, B.x - A.y);
}

#define CANS_SQRT_HALF 0.70710678118654752440

// eq. 2b at one cell from the three face differences; one definition so that every kernel
// that evaluates the divergence rounds identically
CANS_HD double div_value(double du, double dv, double dw, double rdx, double rdy, double rz, double rdt) {
    return (du * rdx + dv * rdy + dw * rz) * rdt;
}

// =================================================================================================
// x pass.  One CTA handles NF row pairs; shared memory: NF lines of P::NPAD cplx.
// =================================================================================================
template <class P, int NF, int NT, int TWOFF = NF * P::NPAD>
struct XPass {
    static constexpr int N = P::N;
    static constexpr int H = N / 2;
    static constexpr int WORK_CPLX = NF * P::NPAD;             // line buffers
    static constexpr int SMEM_CPLX = NF * P::NPAD + P::TW_TOTAL;

    // TWOFF: where this direction's twiddles live relative to the work buffer
    static CANS_HD cplx* tw_smem(cplx* sm) { return sm + TWOFF; }

    static CANS_HD void load_twiddles(const XYArgs& a, cplx* sm, int tid) {
        cplx* t = tw_smem(sm);
        for (int i = tid; i < P::TW_TOTAL; i += NT) t[i] = a.tw[i];
    }

    // pair index -> offset of row a (row b = +nx)
    static CANS_HD size_t row_offset(const XYArgs& a, long pr, int& j, int& k) {
        const int hp = a.ny >> 1;
        const int kl = (int)(pr / hp);
        k = a.k0 + kl;
        j = 2 * (int)(pr - (long)kl * hp);
        return ((size_t)k * a.ny + j) * (size_t)a.nx;
    }

    // ---- forward load (optionally computing the divergence on the fly) ----
    // Loads are issued in batches of UB iterations before the first use, so that every thread keeps
    // 2*UB (22*UB/11 with the divergence) independent 16-byte loads in flight: the load phase is then
    // bound by bandwidth rather than by one memory latency per iteration.
    static constexpr int ITERS = (NF * H + NT - 1) / NT;

    template <bool DIV>
    static CANS_HD void fetch_forward(const XYArgs& a, size_t ro, int j, int k, int e2, double2& va, double2& vb) {
        if (!DIV) {
            va = ld_p2(a.p + ro + 2 * e2);
            vb = ld_p2(a.p + ro + a.nx + 2 * e2);
        } else {
            const size_t plane = (size_t)a.nx * a.ny;
            const int i0 = 2 * e2;
            // u: x differences on rows a and b
            const double2 ua = *reinterpret_cast<const double2*>(a.u + ro + i0);
            const double2 ub = *reinterpret_cast<const double2*>(a.u + ro + a.nx + i0);
            double ula, ulb;
            if (i0 > 0) { ula = a.u[ro + i0 - 1]; ulb = a.u[ro + a.nx + i0 - 1]; }
            else if (a.wrap_x) { ula = a.u[ro + a.nx - 1]; ulb = a.u[ro + 2 * (size_t)a.nx - 1]; }
            else if (a.fx) { ula = a.fx[(size_t)k * a.ny + j]; ulb = a.fx[(size_t)k * a.ny + j + 1]; }
            else { ula = 0.0; ulb = 0.0; }
            // v: rows j-1, j, j+1
            const double2 v1 = *reinterpret_cast<const double2*>(a.v + ro + i0);
            const double2 v2 = *reinterpret_cast<const double2*>(a.v + ro + a.nx + i0);
            double2 v0;
            if (j > 0) v0 = *reinterpret_cast<const double2*>(a.v + ro - a.nx + i0);
            else if (a.wrap_y) v0 = *reinterpret_cast<const double2*>(a.v + ro + (size_t)(a.ny - 1) * a.nx + i0);
            else if (a.fy) v0 = *reinterpret_cast<const double2*>(a.fy + (size_t)k * a.nx + i0);
            else v0 = make_double2(0.0, 0.0);
            // w: planes k-1, k
            const double2 wa = *reinterpret_cast<const double2*>(a.w + ro + i0);
            const double2 wb = *reinterpret_cast<const double2*>(a.w + ro + a.nx + i0);
            double2 wla, wlb;
            if (k > 0) {
                wla = *reinterpret_cast<const double2*>(a.w + ro - plane + i0);
                wlb = *reinterpret_cast<const double2*>(a.w + ro - plane + a.nx + i0);
            } else if (a.wrap_z) {
                wla = *reinterpret_cast<const double2*>(a.w + ro + (size_t)(a.nz - 1) * plane + i0);
                wlb = *reinterpret_cast<const double2*>(a.w + ro + (size_t)(a.nz - 1) * plane + a.nx + i0);
            } else if (a.fz) {
                wla = *reinterpret_cast<const double2*>(a.fz + (size_t)j * a.nx + i0);
                wlb = *reinterpret_cast<const double2*>(a.fz + (size_t)(j + 1) * a.nx + i0);
            } else { wla = make_double2(0.0, 0.0); wlb = wla; }
            const double rz = a.rdzf[k];
            va.x = div_value(ua.x - ula, v1.x - v0.x, wa.x - wla.x, a.rdx, a.rdy, rz, a.rdt);
            va.y = div_value(ua.y - ua.x, v1.y - v0.y, wa.y - wla.y, a.rdx, a.rdy, rz, a.rdt);
            vb.x = div_value(ub.x - ulb, v2.x - v1.x, wb.x - wlb.x, a.rdx, a.rdy, rz, a.rdt);
            vb.y = div_value(ub.y - ub.x, v2.y - v1.y, wb.y - wlb.y, a.rdx, a.rdy, rz, a.rdt);
        }
    }

    template <bool DIV>
    static CANS_HD void load_forward(const XYArgs& a, cplx* sm, long pair0, long npairs, int tid) {
        constexpr int UB = DIV ? (ITERS < 2 ? ITERS : 2) : (ITERS < 8 ? ITERS : 8);
        for (int it0 = 0; it0 < ITERS; it0 += UB) {
            double2 va[UB], vb[UB];
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                const int idx = tid + (it0 + u) * NT;
                const int f = idx / H;
                const int e2 = idx - f * H;
                const long pr = pair0 + f;
                if (idx < NF * H && pr < npairs) {
                    int j, k;
                    const size_t ro = row_offset(a, pr, j, k);
                    fetch_forward<DIV>(a, ro, j, k, e2, va[u], vb[u]);
                }
            }
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                const int idx = tid + (it0 + u) * NT;
                const int f = idx / H;
                const int e2 = idx - f * H;
                if (idx < NF * H && pair0 + f < npairs) {
                    if (kind_mixed(a.kind)) put_forward_mixed(a, sm + f * P::NPAD, e2, va[u], vb[u]);
                    else put_forward(sm + f * P::NPAD, e2, va[u], vb[u], a.kind);
                }
            }
        }
    }

    // samples (2*e2, 2*e2+1) of rows a and b -> FFT input elements of the packed line z = a + i b
    static CANS_HD void put_forward(cplx* line, int e2, double2 va, double2 vb, int kind) {
        cplx z0 = make_double2(va.x, vb.x);      // index 2*e2
        cplx z1 = make_double2(va.y, vb.y);      // index 2*e2+1
        int d0, d1;
        if (kind == KIND_PP) { d0 = 2 * e2; d1 = 2 * e2 + 1; }
        else { d0 = e2; d1 = N - 1 - e2; if (kind_neg_odd(kind)) z1 = cneg(z1); }
        line[P::pad(d0)] = z0;
        line[P::pad(d1)] = z1;
    }
    // the same for the mixed pairs: with the pre-twiddle of the element
    static CANS_HD void put_forward_mixed(const XYArgs& a, cplx* line, int e2, double2 va, double2 vb) {
        const cplx z0 = make_double2(va.x, vb.x);
        cplx z1 = make_double2(va.y, vb.y);
        if (a.kind == KIND_ND) z1 = cneg(z1);
        line[P::pad(e2)] = cmul(z0, a.wpre[e2]);
        line[P::pad(N - 1 - e2)] = cmul(z1, a.wpre[N - 1 - e2]);
    }

    // ---- passes ----
    template <int M, int R, bool INV>
    static CANS_HD void pass(cplx* sm, const cplx* twp, int tid) {
        constexpr int TASKS = N / R;
        for (int t = tid; t < NF * TASKS; t += NT) {
            const int f = t / TASKS;
            const int g = t - f * TASKS;
            cplx* line = sm + f * P::NPAD;
            fft_task<M, R, INV>(line, twp, g, [](int e) { return P::pad(e); });
        }
    }
    static CANS_HD void pass1_fwd(cplx* sm, int tid) { pass<N, P::R1, false>(sm, tw_smem(sm), tid); }
    static CANS_HD void pass2_fwd(cplx* sm, int tid) { if (P::R2 > 1) pass<P::M2, P::R2, false>(sm, tw_smem(sm) + P::TW1, tid); }
    static CANS_HD void pass3_fwd(cplx* sm, int tid) { pass<P::R3, P::R3, false>(sm, nullptr, tid); }
    static CANS_HD void pass1_inv(cplx* sm, int tid) { pass<N, P::R1, true>(sm, tw_smem(sm), tid); }
    static CANS_HD void pass2_inv(cplx* sm, int tid) { if (P::R2 > 1) pass<P::M2, P::R2, true>(sm, tw_smem(sm) + P::TW1, tid); }
    static CANS_HD void pass3_inv(cplx* sm, int tid) { pass<P::R3, P::R3, true>(sm, nullptr, tid); }

    // ---- forward store: separate the two lines and write slots ----
    static CANS_HD void store_forward(const XYArgs& a, const cplx* sm, long pair0, long npairs, int tid) {
        for (int idx = tid; idx < NF * H; idx += NT) {
            const int f = idx / H;
            const int s = idx - f * H;
            const long pr = pair0 + f;
            if (pr >= npairs) continue;
            int j, k;
            const size_t ro = row_offset(a, pr, j, k);
            const cplx* line = sm + f * P::NPAD;
            double2 oa, ob;
            if (kind_mixed(a.kind)) {
                post_forward(line[P::pad(P::loc_of_freq(s))], line[P::pad(P::loc_of_freq(N - 1 - s))], a.wpost[s], a.kind,
                             oa.x, oa.y, ob.x, ob.y);
            } else if (s == 0) {
                const cplx Z0 = line[P::pad(P::loc_of_freq(0))];
                const cplx Zh = line[P::pad(P::loc_of_freq(H))];
                const double c = (a.kind == KIND_PP) ? 1.0 : CANS_SQRT_HALF;
                oa = make_double2(Z0.x, c * Zh.x);
                ob = make_double2(Z0.y, c * Zh.y);
            } else {
                const cplx Zq = line[P::pad(P::loc_of_freq(s))];
                const cplx Zm = line[P::pad(P::loc_of_freq(N - s))];
                cplx wq = make_double2(1.0, 0.0);
                if (a.kind != KIND_PP) wq = a.wpost[s];
                post_forward(Zq, Zm, wq, a.kind, oa.x, oa.y, ob.x, ob.y);
            }
            *reinterpret_cast<double2*>(a.p + ro + 2 * s) = oa;
            *reinterpret_cast<double2*>(a.p + ro + a.nx + 2 * s) = ob;
        }
    }

    // ---- inverse load: slots -> Z at digit-reversed locations (batched like load_forward) ----
    static CANS_HD void load_inverse(const XYArgs& a, cplx* sm, long pair0, long npairs, int tid) {
        constexpr int UB = ITERS < 8 ? ITERS : 8;
        for (int it0 = 0; it0 < ITERS; it0 += UB) {
            double2 ia[UB], ib[UB];
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                const int idx = tid + (it0 + u) * NT;
                const int f = idx / H;
                const int s = idx - f * H;
                const long pr = pair0 + f;
                if (idx < NF * H && pr < npairs) {
                    int j, k;
                    const size_t ro = row_offset(a, pr, j, k);
                    ia[u] = ld_p2(a.p + ro + 2 * s);
                    ib[u] = ld_p2(a.p + ro + a.nx + 2 * s);
                }
            }
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                const int idx = tid + (it0 + u) * NT;
                const int f = idx / H;
                const int s = idx - f * H;
                if (idx < NF * H && pair0 + f < npairs) put_inverse(a, sm + f * P::NPAD, s, ia[u], ib[u]);
            }
        }
    }

    // slot s of rows a and b -> Z at the digit-reversed locations
    static CANS_HD void put_inverse(const XYArgs& a, cplx* line, int s, double2 ia, double2 ib) {
        if (kind_mixed(a.kind)) {
            cplx Zq, Zm;
            pre_inverse(ia.x, ia.y, ib.x, ib.y, a.wpost[s], a.kind, Zq, Zm);
            line[P::pad(P::loc_of_freq(s))] = Zq;
            line[P::pad(P::loc_of_freq(N - 1 - s))] = Zm;
        } else if (s == 0) {
            const double c = (a.kind == KIND_PP) ? 1.0 : (1.0 / CANS_SQRT_HALF);
            line[P::pad(P::loc_of_freq(0))] = make_double2(ia.x, ib.x);
            line[P::pad(P::loc_of_freq(H))] = make_double2(c * ia.y, c * ib.y);
        } else {
            cplx wq = make_double2(1.0, 0.0);
            if (a.kind != KIND_PP) wq = a.wpost[s];
            cplx Zq, Zm;
            pre_inverse(ia.x, ia.y, ib.x, ib.y, wq, a.kind, Zq, Zm);
            line[P::pad(P::loc_of_freq(s))] = Zq;
            line[P::pad(P::loc_of_freq(N - s))] = Zm;
        }
    }

    // ---- inverse store: natural-order z = a + i b back to rows a, b ----
    static CANS_HD void store_inverse(const XYArgs& a, const cplx* sm, long pair0, long npairs, int tid) {
        for (int idx = tid; idx < NF * H; idx += NT) {
            const int f = idx / H;
            const int e2 = idx - f * H;
            const long pr = pair0 + f;
            if (pr >= npairs) continue;
            int j, k;
            const size_t ro = row_offset(a, pr, j, k);
            const cplx* line = sm + f * P::NPAD;
            int d0, d1;
            if (a.kind == KIND_PP) { d0 = 2 * e2; d1 = 2 * e2 + 1; }
            else { d0 = e2; d1 = N - 1 - e2; }
            cplx z0 = line[P::pad(d0)];
            cplx z1 = line[P::pad(d1)];
            if (kind_mixed(a.kind)) { z0 = cmulc(z0, a.wpre[d0]); z1 = cmulc(z1, a.wpre[d1]); }
            if (kind_neg_odd(a.kind)) z1 = cneg(z1);
            *reinterpret_cast<double2*>(a.p + ro + 2 * e2) = make_double2(z0.x, z1.x);
            *reinterpret_cast<double2*>(a.p + ro + a.nx + 2 * e2) = make_double2(z0.y, z1.y);
        }
    }
};

// =================================================================================================
// y pass.  One CTA handles TXC complex columns (2*TXC real columns) of one k-plane, all ny rows;
// shared memory: element (e, f) at e*TXC + f, so every access of 8 consecutive threads is contiguous.
// =================================================================================================
template <class P, int TXC, int NT, int TWOFF = P::N * TXC>
struct YPass {
    static constexpr int N = P::N;
    static constexpr int H = N / 2;
    static constexpr int WORK_CPLX = N * TXC;
    static constexpr int SMEM_CPLX = N * TXC + P::TW_TOTAL;

    static CANS_HD cplx* tw_smem(cplx* sm) { return sm + TWOFF; }
    static CANS_HD void load_twiddles(const XYArgs& a, cplx* sm, int tid) {
        cplx* t = tw_smem(sm);
        for (int i = tid; i < P::TW_TOTAL; i += NT) t[i] = a.tw[i];
    }
    // base = pointer to element (row 0, real column 2*c0) of plane k
    static CANS_HD double* tile_base(const XYArgs& a, int ctile, int k) {
        return a.p + (size_t)k * a.nx * a.ny + 2 * (size_t)ctile * TXC;
    }

    static CANS_HD void load_forward(const XYArgs& a, cplx* sm, int ctile, int k, int tid) {
        const double* base = tile_base(a, ctile, k);
        constexpr int ITERS = (N * TXC + NT - 1) / NT;
        constexpr int UB = ITERS < 12 ? ITERS : 12;        // independent 16-byte loads in flight per thread
        for (int it0 = 0; it0 < ITERS; it0 += UB) {
            cplx z[UB];
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                const int idx = tid + (it0 + u) * NT;
                const int j = idx / TXC;
                const int f = idx - j * TXC;
                if (idx < N * TXC) z[u] = ld_p2(base + (size_t)j * a.nx + 2 * f);
            }
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                const int idx = tid + (it0 + u) * NT;
                const int j = idx / TXC;
                const int f = idx - j * TXC;
                if (idx < N * TXC) put_forward(a, sm, j, f, z[u]);
            }
        }
    }

    static CANS_HD void put_forward(const XYArgs& a, cplx* sm, int j, int f, cplx z) {
        const int e = elem_of_index<N>(j, a.kind);
        if (kind_neg_odd(a.kind) && (j & 1)) z = cneg(z);
        if (kind_mixed(a.kind)) z = cmul(z, a.wpre[e]);
        sm[e * TXC + f] = z;
    }

    template <int M, int R, bool INV>
    static CANS_HD void pass(cplx* sm, const cplx* twp, int tid) {
        constexpr int TASKS = N / R;
        for (int t = tid; t < TXC * TASKS; t += NT) {
            const int g = t / TXC;
            const int f = t - g * TXC;
            fft_task<M, R, INV>(sm, twp, g, [f](int e) { return e * TXC + f; });
        }
    }
    static CANS_HD void pass1_fwd(cplx* sm, int tid) { pass<N, P::R1, false>(sm, tw_smem(sm), tid); }
    static CANS_HD void pass2_fwd(cplx* sm, int tid) { if (P::R2 > 1) pass<P::M2, P::R2, false>(sm, tw_smem(sm) + P::TW1, tid); }
    static CANS_HD void pass3_fwd(cplx* sm, int tid) { pass<P::R3, P::R3, false>(sm, nullptr, tid); }
    static CANS_HD void pass1_inv(cplx* sm, int tid) { pass<N, P::R1, true>(sm, tw_smem(sm), tid); }
    static CANS_HD void pass2_inv(cplx* sm, int tid) { if (P::R2 > 1) pass<P::M2, P::R2, true>(sm, tw_smem(sm) + P::TW1, tid); }
    static CANS_HD void pass3_inv(cplx* sm, int tid) { pass<P::R3, P::R3, true>(sm, nullptr, tid); }

    static CANS_HD void store_forward(const XYArgs& a, const cplx* sm, int ctile, int k, int tid) {
        double* base = tile_base(a, ctile, k);
        for (int idx = tid; idx < H * TXC; idx += NT) {
            const int s = idx / TXC;
            const int f = idx - s * TXC;
            double2 r0, r1;   // rows 2s and 2s+1: (column a, column b)
            if (kind_mixed(a.kind)) {
                double A0, A1, B0, B1;
                post_forward(sm[P::loc_of_freq(s) * TXC + f], sm[P::loc_of_freq(N - 1 - s) * TXC + f], a.wpost[s], a.kind,
                             A0, A1, B0, B1);
                r0 = make_double2(A0, B0);
                r1 = make_double2(A1, B1);
            } else if (s == 0) {
                const cplx Z0 = sm[P::loc_of_freq(0) * TXC + f];
                const cplx Zh = sm[P::loc_of_freq(H) * TXC + f];
                const double c = (a.kind == KIND_PP) ? 1.0 : CANS_SQRT_HALF;
                r0 = make_double2(Z0.x, Z0.y);
                r1 = make_double2(c * Zh.x, c * Zh.y);
            } else {
                const cplx Zq = sm[P::loc_of_freq(s) * TXC + f];
                const cplx Zm = sm[P::loc_of_freq(N - s) * TXC + f];
                cplx wq = make_double2(1.0, 0.0);
                if (a.kind != KIND_PP) wq = a.wpost[s];
                double A0, A1, B0, B1;
                post_forward(Zq, Zm, wq, a.kind, A0, A1, B0, B1);
                r0 = make_double2(A0, B0);
                r1 = make_double2(A1, B1);
            }
            *reinterpret_cast<double2*>(base + (size_t)(2 * s) * a.nx + 2 * f) = r0;
            *reinterpret_cast<double2*>(base + (size_t)(2 * s + 1) * a.nx + 2 * f) = r1;
        }
    }

    static CANS_HD void load_inverse(const XYArgs& a, cplx* sm, int ctile, int k, int tid) {
        const double* base = tile_base(a, ctile, k);
        constexpr int ITERS = (H * TXC + NT - 1) / NT;
        constexpr int UB = ITERS < 6 ? ITERS : 6;
        for (int it0 = 0; it0 < ITERS; it0 += UB) {
            double2 r0[UB], r1[UB];
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                const int idx = tid + (it0 + u) * NT;
                const int s = idx / TXC;
                const int f = idx - s * TXC;
                if (idx < H * TXC) {
                    r0[u] = ld_p2(base + (size_t)(2 * s) * a.nx + 2 * f);
                    r1[u] = ld_p2(base + (size_t)(2 * s + 1) * a.nx + 2 * f);
                }
            }
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                const int idx = tid + (it0 + u) * NT;
                const int s = idx / TXC;
                const int f = idx - s * TXC;
                if (idx < H * TXC) put_inverse(a, sm, s, f, r0[u], r1[u]);
            }
        }
    }

    static CANS_HD void put_inverse(const XYArgs& a, cplx* sm, int s, int f, double2 r0, double2 r1) {
        if (kind_mixed(a.kind)) {
            cplx Zq, Zm;
            pre_inverse(r0.x, r1.x, r0.y, r1.y, a.wpost[s], a.kind, Zq, Zm);
            sm[P::loc_of_freq(s) * TXC + f] = Zq;
            sm[P::loc_of_freq(N - 1 - s) * TXC + f] = Zm;
        } else if (s == 0) {
            const double c = (a.kind == KIND_PP) ? 1.0 : (1.0 / CANS_SQRT_HALF);
            sm[P::loc_of_freq(0) * TXC + f] = make_double2(r0.x, r0.y);
            sm[P::loc_of_freq(H) * TXC + f] = make_double2(c * r1.x, c * r1.y);
        } else {
            cplx wq = make_double2(1.0, 0.0);
            if (a.kind != KIND_PP) wq = a.wpost[s];
            cplx Zq, Zm;
            pre_inverse(r0.x, r1.x, r0.y, r1.y, wq, a.kind, Zq, Zm);
            sm[P::loc_of_freq(s) * TXC + f] = Zq;
            sm[P::loc_of_freq(N - s) * TXC + f] = Zm;
        }
    }

    static CANS_HD void store_inverse(const XYArgs& a, const cplx* sm, int ctile, int k, int tid) {
        double* base = tile_base(a, ctile, k);
        for (int idx = tid; idx < N * TXC; idx += NT) {
            const int j = idx / TXC;
            const int f = idx - j * TXC;
            const int e = elem_of_index<N>(j, a.kind);
            cplx z = sm[e * TXC + f];
            if (kind_mixed(a.kind)) z = cmulc(z, a.wpre[e]);
            if (kind_neg_odd(a.kind) && (j & 1)) z = cneg(z);
            *reinterpret_cast<double2*>(base + (size_t)j * a.nx + 2 * f) = z;
        }
    }
};

}  // namespace cans
