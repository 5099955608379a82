// z_pass.cuh -- the tridiagonal solve along z for every (kx, ky) mode: eq. 6, "solved very
// efficiently with Gauss elimination", on a possibly non-uniform z grid.
//
//   (b_k + lam) x_k + a_k x_{k-1} + c_k x_{k+1} = d_k ,   lam = lam_x(i)/dx^2 + lam_y(j)/dy^2 <= 0
//
// Thomas recurrence (same algebra as the sequential algorithm):
//   r_k = 1 / (b_k + lam - a_k c_{k-1} r_{k-1}),  d'_k = (d_k - a_k d'_{k-1}) r_k,  x_k = d'_k - c_k r_k x_{k+1}
//
// B200 mapping ("register-resident partitioned Thomas", fed by an asynchronous tile pipeline):
//   * a CTA is persistent and draws tiles of TC consecutive columns (x fastest => TC*8 contiguous
//     bytes per row) from a global ticket counter; the tile of the NEXT ticket is copied global ->
//     shared by the TMA unit (one cp.async.bulk.tensor.2d per box, completion on an mbarrier; z_solve.cu)
//     while the current tile is being solved, so HBM reads stay in flight during the whole arithmetic phase;
//   * a column is cut into P segments of MROWS rows; thread (c, s) owns segment s of column c with
//     its MROWS right-hand sides in registers; the whole column never leaves the SM between the
//     forward and backward sweeps (16 B/cell of HBM traffic, the structural minimum);
//   * the pivot chain r_k is restarted at every segment from a plan-time table r_{k0-1}(mode, s)
//     (nx*ny*P doubles, 1/MROWS of a field) and recomputed in-register -- bit-identical to the
//     sequential pivots;
//   * d' and x are first-order linear recurrences: each segment runs them from a zero start while
//     accumulating the propagation factor (prod of -a_k r_k, resp. -c_k r_k); a scan over the segment ends --
//     composed per warp by shuffles, one aggregate per group of 32/TC segments in shared memory (group_scan) --
//     supplies the true start value, which is then propagated;
//   * results go straight from registers to global memory (coalesced rows, a walking pointer, no per-row predicate).
// The singular kx = ky = 0 column of an all-periodic/Neumann problem is handled by z_singular_stage / _sweeps / _store
// (CTA 0, before it joins the tile loop).
//
// Periodic z (the triperiodic Taylor-Green case of P:L222): the system is cyclic, row 0 couples to
// x_{nz-1} through a_0 and row nz-1 to x_0 through c_{nz-1}.  Sherman-Morrison on the same partitioned Thomas: with
// gamma = -(b_0 + lam), the open matrix T' = T - u v^T (u = (gamma, 0, .., 0, c_{nz-1}), v = (1, 0, .., 0, a_0/gamma))
// has b'_0 = 2 (b_0 + lam) and b'_{nz-1} = b_{nz-1} + lam + c_{nz-1} a_0 / (b_0 + lam).  T' q = u and T' y = d share the
// pivots AND the propagation factors of both sweeps, so q rides along in the same three phases: its forward values cost
// one FMA per row, its rows live in the tile's own staging buffer (free once the right-hand side is in registers), and
// x = y - q (y_0 + v_n y_{nz-1}) / (1 + q_0 + v_n q_{nz-1}) is formed in the final store loop (one more CTA barrier
// than the open system, for the four edge values of each column).
#pragma once
#include "common.cuh"

namespace cans {

struct ZArgs {
    int nx, ny, nz;
    int nseg;                 // P = ceil(nz / MROWS)
    long ncols;               // nx * ny
    long ntiles;              // ceil(ncols / TC)
    double* p;                // field, solved in place
    const double* lamx;       // [nx]  lam_x(position)/dx^2
    const double* lamy;       // [ny]  lam_y(position)/dy^2
    const double* az;         // [nseg*MROWS] sub-diagonal a_k        (0 beyond nz, a_0 = 0)
    const double* bz;         // diagonal b_k with boundary rows folded in (-1 beyond nz: keeps the padded pivots finite)
    const double* cz;         // super-diagonal c_k                   (0 beyond nz, c_{nz-1} = 0)
    const double* gz;         // a_k * c_{k-1}                        (0 for k = 0 and beyond nz)
    const double* rstart;     // [nseg][ncols]  r_{s*MROWS-1}(column)  (0 for s = 0)
    double scale;             // 1/(nx*ny): normalisation of the two unnormalised inverse FFTs
    int singular;             // 1: column 0 is the singular mode, skipped by the tile path
    const double* r00;        // [nz] pivots of the singular column (rows 0..nz-2), plan-time
    const double* dzf;        // [nz]
    double inv_lz;            // 1 / sum(dzf)
    unsigned int* ticket;     // tile ticket counter (zeroed before the launch)
    double alpha;             // Helmholtz shift added to every eigenvalue (eq. 3b): (L + alpha I) Phi = f; 0 for eq. 5
    int nz_solve;             // rows [0, nz_solve) form the tridiagonal system; rows [nz_solve, nz) are passed through
                              // (scaled): the wall slot of a face-located unknown (nz_solve = nz - 1), else nz_solve = nz
    int cyclic;               // 1: z is periodic (az[0] = cz[nz-1] = 0 in the tables, the wrap couplings are below)
    double a0w, cw;           // a_0 = 1/(dzf_0 dzc_0) and c_{nz-1} = 1/(dzf_{nz-1} dzc_nz) of the cyclic system
    unsigned long long nx_magic;   // ceil(2^40 / nx): j = (col * nx_magic) >> 40 is col / nx exactly for col < nx*ny <= 2^22
    int nbox, box_rows;       // TMA tiling of a column tile: nbox boxes of box_rows rows (set by z_solve_launch)
};

// one pivot step; shared by the plan-time table kernel and the solve so the values are identical
// The reciprocal is the hardware seed (rcp.approx, ~20 bits) refined by two Newton steps: full double precision
// to about one unit in the last place for these well-scaled, strictly negative denominators, without the range
// checks and the slow path of the IEEE division -- the pivot chain is the longest dependency chain of the solve.
CANS_HD double z_pivot_bl(double bl, double gk, double rprev) {
    const double den = bl - gk * rprev;
#if defined(__CUDA_ARCH__)
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(den));
    r = fma(fma(-den, r, 1.0), r, r);
    r = fma(fma(-den, r, 1.0), r, r);
    return r;
#else
    return 1.0 / den;
#endif
}
CANS_HD double z_pivot(double bk, double lam, double gk, double rprev) { return z_pivot_bl(bk + lam, gk, rprev); }

// diagonal entry of row k of the cyclic system's open matrix T' (b0 = table entry of row 0)
CANS_HD double z_cyclic_diag(const ZArgs& a, int k, double bk, double b0, double lam) {
    double bl = bk + lam;
    if (k == 0) bl += bl;
    if (k == a.nz - 1) bl += a.cw * a.a0w / (b0 + lam);
    return bl;
}

template <int MROWS>
struct ZState {
    double d[MROWS];
    double r[MROWS];
    double start;     // true d'_{k0-1}, later true x_{k0+MROWS}
    double startq;    // the same for the correction vector q of a cyclic system
    double exe, exf, exq;   // composition of the warp's earlier (forward) / later (backward) segments of this column:
                            // value -> exe + exf * value (exq: the end term of q), see group_scan
    long col;
    bool active;
};

// shared memory (doubles): tables az [nzp], (bz, gz) pairs [2 nzp], cz [nzp]; (end, factor) pairs of the forward sweep [TC*P] and a second
// array for the backward sweep (so that no barrier is needed between reading one and writing the other); the same two
// arrays of segment ends for q [TC*P] each; (y_0, q_0, y_{nz-1}, q_{nz-1}) per column of a cyclic solve [4*TC]; two tile
// buffers [nzp][TC]
template <int MROWS, int TC>
struct ZPass {
    static CANS_HD size_t scan_offset(int nseg) { return (size_t)4 * nseg * MROWS; }
    static CANS_HD size_t scanq_offset(int nseg) { return scan_offset(nseg) + (size_t)4 * TC * nseg; }
    static CANS_HD size_t edge_offset(int nseg) { return scanq_offset(nseg) + (size_t)2 * TC * nseg; }
    // (rounded up to 1 KB so that the tile buffers the TMA unit fills start on a 1 KB boundary)
    static CANS_HD size_t table_doubles(int nseg) { return (edge_offset(nseg) + 4 * TC + 127) / 128 * 128; }
    static CANS_HD size_t tile_doubles(int nseg) { return (size_t)nseg * MROWS * TC; }
    static CANS_HD size_t smem_doubles(int nseg) { return table_doubles(nseg) + 2 * tile_doubles(nseg); }

    static CANS_HD void load_tables(const ZArgs& a, double* sm, int tid, int nthreads) {
        const int nzp = a.nseg * MROWS;
        // az [nzp] | (bz, gz) pairs [nzp] (phase 1 reads both with one 16-byte load) | cz [nzp]
        for (int i = tid; i < nzp; i += nthreads) {
            sm[i] = a.az[i];
            sm[nzp + 2 * i] = a.bz[i];
            sm[nzp + 2 * i + 1] = a.gz[i];
            sm[3 * nzp + i] = a.cz[i];
        }
    }

    // Segment scans.  The true start of a segment is the composition of the affine maps x -> end + factor * x of all the
    // segments before it (forward sweep) or above it (backward sweep).  A warp holds G = 32 / TC consecutive segments of
    // its columns (lanes c + TC * sg): it composes those by shuffles, publishes ONE aggregate per group and keeps each
    // lane's in-group prefix in registers, so the serial scan behind the barrier walks groups, not segments -- half
    // (TC = 16) or a quarter (TC = 8) of the 16-byte shared-memory reads and of the dependent steps.
    static constexpr int G = 32 / TC;
    // does the warp of segment s hold the segment of row nz-1 ?  (warp-uniform)
    static CANS_HD bool last_group(const ZArgs& a, int s) { return s / G == ((a.nz - 1) / MROWS) / G; }
    static CANS_HD int ngroups(int nseg) { return (nseg + G - 1) / G; }
    // DOWN = false: compose with the earlier segments (lanes below); true: with the later ones (lanes above).
    // In: this segment's (e, f, q).  Out: (e, f, q) = aggregate of the group as seen from its last (first) lane;
    // (xe, xf, xq) = composition of the in-group segments before (after) this lane, identity if none.
    template <bool CYC, bool DOWN>
    static CANS_HD void group_scan(int tid, int s, int nseg, double& e, double& f, double& q, double& xe, double& xf, double& xq) {
        xe = 0.0; xf = 1.0; xq = 0.0;
        if (G == 1) return;
#if defined(__CUDA_ARCH__)
        // the lanes of this warp that exist (the last warp of a CTA of TC * nseg threads may be partial)
        const int left = TC * nseg - (tid & ~31);
        const unsigned mask = left >= 32 ? 0xffffffffu : ((1u << left) - 1u);
        const int sg = s % G;
#pragma unroll
        for (int off = 1; off < G; off <<= 1) {
            const double e2 = DOWN ? __shfl_down_sync(mask, e, off * TC) : __shfl_up_sync(mask, e, off * TC);
            const double f2 = DOWN ? __shfl_down_sync(mask, f, off * TC) : __shfl_up_sync(mask, f, off * TC);
            double q2 = 0.0;
            if (CYC) q2 = DOWN ? __shfl_down_sync(mask, q, off * TC) : __shfl_up_sync(mask, q, off * TC);
            const bool has = DOWN ? (sg + off < G && s + off < nseg) : (sg >= off);
            if (has) { e = e + f * e2; if (CYC) q = q + f * q2; f = f * f2; }
        }
        const double e1 = DOWN ? __shfl_down_sync(mask, e, TC) : __shfl_up_sync(mask, e, TC);
        const double f1 = DOWN ? __shfl_down_sync(mask, f, TC) : __shfl_up_sync(mask, f, TC);
        double q1 = 0.0;
        if (CYC) q1 = DOWN ? __shfl_down_sync(mask, q, TC) : __shfl_up_sync(mask, q, TC);
        const bool has1 = DOWN ? (sg + 1 < G && s + 1 < nseg) : (sg >= 1);
        if (has1) { xe = e1; xf = f1; xq = q1; }
#endif
    }

    // The two rows in which the open matrix T' and the right-hand side u of the correction system differ from the plain
    // tridiagonal rows, as seen by the thread of segment s: row 0 (diagonal doubled, u_0 = gamma = -(b_0 + lam)) and row
    // nz-1 (diagonal + c_{nz-1} a_0 / (b_0 + lam), u_{nz-1} = c_{nz-1}).
    struct CyclicRows {
        double diag0 = 0.0, rhs0 = 0.0, diagn = 0.0;
        int rl = -1;
    };
    static CANS_HD CyclicRows cyclic_rows(const ZArgs& a, double b0, double lam, int s) {
        CyclicRows cr;
        const double bl0 = b0 + lam;
        if (s == 0) { cr.diag0 = bl0; cr.rhs0 = -bl0; }
        if (s == (a.nz - 1) / MROWS) { cr.rl = (a.nz - 1) - s * MROWS; cr.diagn = a.cw * a.a0w / bl0; }
        return cr;
    }

    // the rows of phase 1 (CYC: cyclic system; LAST: this thread's segment holds row nz-1, at local row cr.rl)
    template <bool CYC, bool LAST>
    static CANS_HD void phase1_rows(const ZArgs& a, const double* saz, const double2* sbg, ZState<MROWS>& st,
                                    int k0, double rstart_val, double lam, const CyclicRows& cr, double& dp_out, double& fac_out,
                                    double& dq_out) {
        double rp = rstart_val;
        double dp = 0.0, fac = 1.0, dq = 0.0;
#pragma unroll
        for (int r = 0; r < MROWS; ++r) {
            const int k = k0 + r;
            const double2 bg = sbg[k];
            double bl = bg.x + lam;
            if (CYC && r == 0) bl += cr.diag0;
            if (LAST && r == cr.rl) bl += cr.diagn;
            rp = z_pivot_bl(bl, bg.y, rp);
            st.r[r] = rp;
            const double e = saz[k] * rp;
            dp = st.d[r] * rp - e * dp;
            st.d[r] = dp;
            fac *= -e;
            if (CYC) {
                if (r == 0) dq = cr.rhs0 * rp;             // zero start; rhs0 = gamma in segment 0, 0 elsewhere
                else dq = -e * dq;
                if (LAST && r == cr.rl) dq = fma(a.cw, rp, dq);
            }
        }
        dp_out = dp; fac_out = fac; dq_out = dq;
    }
    // the rows of phase 2b
    template <bool CYC, bool LAST>
    static CANS_HD void phase2b_rows(const ZArgs& a, const double* saz, const double* scz, ZState<MROWS>& st, int k0,
                                     const CyclicRows& cr, double* qcol, double& xs_out, double& g_out, double& xq_out) {
        double fac = 1.0;
        const double D = st.start;
        double dq = st.startq;
#pragma unroll
        for (int r = 0; r < MROWS; ++r) {
            const double e = saz[k0 + r] * st.r[r];
            fac *= -e;
            st.d[r] += fac * D;
            if (CYC) {
                dq = -e * dq;
                if (r == 0) dq = fma(cr.rhs0, st.r[r], dq);
                if (LAST && r == cr.rl) dq = fma(a.cw, st.r[r], dq);
                qcol[r * TC] = dq;
            }
        }
        double xs = 0.0, g = 1.0, xq = 0.0;
#pragma unroll
        for (int r = MROWS - 1; r >= 0; --r) {
            const double cp = scz[k0 + r] * st.r[r];
            xs = st.d[r] - cp * xs;
            st.d[r] = xs;
            g *= -cp;
            if (CYC) {
                xq = qcol[r * TC] - cp * xq;
                qcol[r * TC] = xq;
            }
        }
        xs_out = xs; g_out = g; xq_out = xq;
    }

    // phase 1: take the segment from the tile buffer, pivots, local forward sweep from a zero start; publish (end, factor)
    // -- and, for a cyclic system, the end of q's local forward sweep
    template <bool CYC>
    static CANS_HD void phase1(const ZArgs& a, double* sm, const double* buf, ZState<MROWS>& st, long tile,
                               double rstart_val, double lam, int tid) {
        const int nzp = a.nseg * MROWS;
        const double* saz = sm;
        const double2* sbg = reinterpret_cast<const double2*>(sm + nzp);
        double2* s_scan = reinterpret_cast<double2*>(sm + scan_offset(a.nseg));      // forward (end, factor) pairs
        double* s_scanq = sm + scanq_offset(a.nseg);
        const int c = tid % TC;
        const int s = tid / TC;
        const long col = tile * TC + c;
        st.col = col;
        st.active = (col < a.ncols) && !(a.singular && col == 0);
        const int k0 = s * MROWS;
        double dp = 0.0, fac = 0.0, dq = 0.0;
        if (col < a.ncols) {
            // (rows nz..nzp-1 of the buffer lie outside the tensor: the TMA unit filled them with zeros)
#pragma unroll
            for (int r = 0; r < MROWS; ++r) st.d[r] = buf[(size_t)(k0 + r) * TC + c] * a.scale;
            if (!CYC) {
                phase1_rows<false, false>(a, saz, sbg, st, k0, rstart_val, lam, CyclicRows(), dp, fac, dq);
            } else {
                // cyclic system: only rows 0 and nz-1 differ from the open one -- row 0 belongs to segment 0 (r = 0 at
                // compile time), row nz-1 to local row rl of the last segment: its threads run their own copy of the loop
                const CyclicRows cr = cyclic_rows(a, sbg[0].x, lam, s);
                // (the choice is made per warp -- the warp holding the last segment runs the general copy in all its lanes,
                // rl = -1 matching no row -- so that no warp executes both copies)
                if (!last_group(a, s)) phase1_rows<true, false>(a, saz, sbg, st, k0, rstart_val, lam, cr, dp, fac, dq);
                else phase1_rows<true, true>(a, saz, sbg, st, k0, rstart_val, lam, cr, dp, fac, dq);
            }
        }
        // compose the warp's segments; the last lane of each group publishes its aggregate
        group_scan<CYC, false>(tid, s, a.nseg, dp, fac, dq, st.exe, st.exf, st.exq);
        if (s % G == G - 1 || s == a.nseg - 1) {
            s_scan[(s / G) * TC + c] = make_double2(dp, fac);
            if (CYC) s_scanq[(s / G) * TC + c] = dq;
        }
    }

    // phase 2: scan the segment ends -> true start; propagate; local backward sweep from a zero start; publish
    template <bool CYC>
    static CANS_HD void phase2a(const ZArgs& a, double* sm, ZState<MROWS>& st, int tid) {
        const double2* s_scan = reinterpret_cast<const double2*>(sm + scan_offset(a.nseg));
        const double* s_scanq = sm + scanq_offset(a.nseg);
        const int c = tid % TC;
        const int s = tid / TC;
        double D = 0.0, Dq = 0.0;           // true d' (and q's) at the end of the previous group ...
        const int grp = s / G;
#pragma unroll 4
        for (int q = 0; q < grp; ++q) {
            const double2 ef = s_scan[q * TC + c];      // one 16-byte load per group
            if (CYC) Dq = s_scanq[q * TC + c] + ef.y * Dq;
            D = ef.x + ef.y * D;
        }
        st.start = st.exe + st.exf * D;     // ... carried through the warp's earlier segments of this group
        st.startq = st.exq + st.exf * Dq;
    }
    // (2b publishes into the backward arrays, so 2a and 2b need no barrier between them).  Cyclic: q's true forward values
    // are rebuilt row by row from its true start and parked in qbuf, then swept backwards in place.
    template <bool CYC>
    static CANS_HD void phase2b(const ZArgs& a, double* sm, ZState<MROWS>& st, double lam, int tid, double* qbuf) {
        const int nzp = a.nseg * MROWS;
        const double* saz = sm;
        const double* scz = sm + 3 * nzp;
        double2* s_scan = reinterpret_cast<double2*>(sm + scan_offset(a.nseg)) + TC * a.nseg;   // backward pairs
        double* s_scanq = sm + scanq_offset(a.nseg) + TC * a.nseg;
        const int c = tid % TC;
        const int s = tid / TC;
        const int k0 = s * MROWS;
        double xs = 0.0, g = 0.0, xq = 0.0;
        if (st.col < a.ncols) {
            double* qcol = qbuf + (size_t)k0 * TC + c;      // this thread's rows of q: qcol[r * TC]
            if (!CYC) {
                phase2b_rows<false, false>(a, saz, scz, st, k0, CyclicRows(), qcol, xs, g, xq);
            } else {
                const CyclicRows cr = cyclic_rows(a, sm[nzp], lam, s);
                if (!last_group(a, s)) phase2b_rows<true, false>(a, saz, scz, st, k0, cr, qcol, xs, g, xq);
                else phase2b_rows<true, true>(a, saz, scz, st, k0, cr, qcol, xs, g, xq);
            }
        }
        // (xs, g): x^0 at the top row of the segment and its factor; compose the warp's segments from the top down, the
        // first lane of each group publishes its aggregate
        group_scan<CYC, true>(tid, s, a.nseg, xs, g, xq, st.exe, st.exf, st.exq);
        if (s % G == 0) {
            s_scan[(s / G) * TC + c] = make_double2(xs, g);
            if (CYC) s_scanq[(s / G) * TC + c] = xq;
        }
    }

    // phase 3 of the open system: scan from the bottom -> true x below the segment; propagate; store to the field
    static CANS_HD void phase3(const ZArgs& a, double* sm, ZState<MROWS>& st, int tid, const double* buf) {
        const int nzp = a.nseg * MROWS;
        const double* scz = sm + 3 * nzp;
        const double2* s_scan = reinterpret_cast<const double2*>(sm + scan_offset(a.nseg)) + TC * a.nseg;   // backward pairs
        const int c = tid % TC;
        const int s = tid / TC;
        const int k0 = s * MROWS;
        double X = 0.0;                     // true x at the top row of the next group ...
#pragma unroll 4
        for (int q = ngroups(a.nseg) - 1; q > s / G; --q) {
            const double2 ef = s_scan[q * TC + c];
            X = ef.x + ef.y * X;
        }
        X = st.exe + st.exf * X;            // ... carried down through the warp's later segments of this group
        if (st.active) {
            const size_t plane = (size_t)a.ncols;
            double g = 1.0;
#pragma unroll
            for (int r = MROWS - 1; r >= 0; --r) {
                g *= -(scz[k0 + r] * st.r[r]);
                st.d[r] += g * X;
            }
            double* out = a.p + (size_t)k0 * plane + st.col;
            if (k0 + MROWS <= a.nz_solve) {                 // whole segment inside the system (warp-uniform)
#pragma unroll
                for (int r = 0; r < MROWS; ++r) out[(size_t)r * plane] = st.d[r];
            } else {
#pragma unroll
                for (int r = 0; r < MROWS; ++r) {
                    const int k = k0 + r;
                    // (the tile buffer still holds this tile: its buffer is not refilled before the next iteration)
                    if (k < a.nz) out[(size_t)r * plane] = (k < a.nz_solve) ? st.d[r] : buf[(size_t)k * TC + c] * a.scale;
                }
            }
        }
    }

    // phase 3 of a cyclic system, first half: the backward scans of y and q; the threads holding rows 0 and nz-1 publish
    // the true (y_0, q_0) and (y_{nz-1}, q_{nz-1}) of their column
    static CANS_HD void cyclic_scan(const ZArgs& a, double* sm, ZState<MROWS>& st, int tid, const double* qbuf) {
        const double2* s_scan = reinterpret_cast<const double2*>(sm + scan_offset(a.nseg)) + TC * a.nseg;
        const double* s_scanq = sm + scanq_offset(a.nseg) + TC * a.nseg;
        double* edge = sm + edge_offset(a.nseg);
        const int c = tid % TC;
        const int s = tid / TC;
        double X = 0.0, Xq = 0.0;
#pragma unroll 4
        for (int q = ngroups(a.nseg) - 1; q > s / G; --q) {
            const double2 ef = s_scan[q * TC + c];
            Xq = s_scanq[q * TC + c] + ef.y * Xq;
            X = ef.x + ef.y * X;
        }
        Xq = st.exq + st.exf * Xq;
        X = st.exe + st.exf * X;
        st.start = X;
        st.startq = Xq;
        if (st.col < a.ncols) {
            if (s == 0) {                                   // row 0: local value + (factor of the whole segment) * X
                const double* scz0 = sm + 3 * a.nseg * MROWS;
                double g = 1.0;
#pragma unroll
                for (int r = 0; r < MROWS; ++r) g *= -(scz0[r] * st.r[r]);
                edge[4 * c] = st.d[0] + g * X;
                edge[4 * c + 1] = qbuf[c] + g * Xq;
            }
            if (s == (a.nz - 1) / MROWS) {                  // row nz-1: last segment, nothing above it: local = true
                double yn = 0.0;
#pragma unroll
                for (int r = 0; r < MROWS; ++r) if (s * MROWS + r == a.nz - 1) yn = st.d[r];
                edge[4 * c + 2] = yn;
                edge[4 * c + 3] = qbuf[(size_t)(a.nz - 1) * TC + c];
            }
        }
    }
    // ... second half (behind a barrier): x = y - q (y_0 + v y_n) / (1 + q_0 + v q_n), v = a_0 / gamma, with the
    // propagation of both backward sweeps folded into one term
    static CANS_HD void cyclic_store(const ZArgs& a, double* sm, ZState<MROWS>& st, double lam, int tid, const double* qbuf) {
        if (!st.active) return;
        const double* edge = sm + edge_offset(a.nseg);
        const int nzp = a.nseg * MROWS;
        const double* scz = sm + 3 * nzp;
        const int c = tid % TC;
        const int k0 = (tid / TC) * MROWS;
        const double v = a.a0w / -(sm[nzp] + lam);                     // sm[nzp] = bz[0]
        const double fact = (edge[4 * c] + v * edge[4 * c + 2]) / (1.0 + edge[4 * c + 1] + v * edge[4 * c + 3]);
        const double Xc = st.start - st.startq * fact;
        const double* qcol = qbuf + (size_t)k0 * TC + c;
        double g = 1.0;
#pragma unroll
        for (int r = MROWS - 1; r >= 0; --r) {
            g *= -(scz[k0 + r] * st.r[r]);
            st.d[r] = (st.d[r] - qcol[r * TC] * fact) + g * Xc;
        }
        const size_t plane = (size_t)a.ncols;
        double* out = a.p + (size_t)k0 * plane + st.col;
        if (k0 + MROWS <= a.nz) {                           // whole segment inside the field (warp-uniform)
#pragma unroll
            for (int r = 0; r < MROWS; ++r) out[(size_t)r * plane] = st.d[r];
        } else {
#pragma unroll
            for (int r = 0; r < MROWS; ++r) if (k0 + r < a.nz) out[(size_t)r * plane] = st.d[r];
        }
    }
};

// plan-time: pivots at the segment boundaries of every column (thread per column, sequential in k)
template <int MROWS>
CANS_HD void z_setup_column(const ZArgs& a, double* rstart_out, double* r00_out, long col) {
    const int i = (int)(col % a.nx);
    const int j = (int)(col / a.nx);
    const double lam = a.lamx[i] + a.lamy[j] + a.alpha;
    double rp = 0.0;
    const int nzp = a.nseg * MROWS;
    for (int k = 0; k < nzp; ++k) {
        if (k % MROWS == 0) rstart_out[(size_t)(k / MROWS) * a.ncols + col] = rp;
        if (a.cyclic) rp = z_pivot_bl(z_cyclic_diag(a, k, a.bz[k], a.bz[0], lam), a.gz[k], rp);
        else rp = z_pivot(a.bz[k], lam, a.gz[k], rp);
        if (col == 0 && k < a.nz && r00_out && !a.cyclic) r00_out[k] = rp;
    }
    if (col == 0 && r00_out && a.cyclic) {
        // singular column of a periodic-z problem: the open system of rows 0..nz-2 with the unmodified diagonal
        rp = 0.0;
        for (int k = 0; k < a.nz; ++k) { rp = z_pivot(a.bz[k], 0.0, a.gz[k], rp); r00_out[k] = rp; }
    }
}

// The singular column (reading S3 / oracle O4): forward sweep on rows 0..nz-2, x[nz-1] = 0, back-substitute, subtract the
// dzf-weighted mean.  The CTA stages t_k = d_k r_k, e_k = a_k r_k, cp_k = c_k r_k and dzf in shared memory in parallel
// (z_singular_stage), ONE thread runs the two recurrences -- one dependent FMA per row -- and leaves the mean in sd[nz]
// (z_singular_sweeps), and the CTA writes the column back (z_singular_store).  sd: 4 * nzp + 1 doubles.
CANS_HD void z_singular_stage(const ZArgs& a, double* sd, int nzp, int tid, int nthreads) {
    for (int k = tid; k < a.nz; k += nthreads) {
        const double rk = a.r00[k];
        sd[k] = a.p[(size_t)k * a.ncols] * a.scale * rk;
        sd[nzp + k] = a.az[k] * rk;
        sd[2 * nzp + k] = a.cz[k] * rk;
        sd[3 * nzp + k] = a.dzf[k];
    }
}
CANS_HD void z_singular_sweeps(const ZArgs& a, double* sd, int nzp) {
    const int nz = a.nz;
    const double* se = sd + nzp;
    const double* scp = sd + 2 * nzp;
    const double* sw = sd + 3 * nzp;
    double dp = 0.0;
#pragma unroll 8
    for (int k = 0; k < nz - 1; ++k) {
        dp = sd[k] - se[k] * dp;
        sd[k] = dp;
    }
    double x = 0.0, acc = 0.0;
    sd[nz - 1] = 0.0;
#pragma unroll 8
    for (int k = nz - 2; k >= 0; --k) {
        x = sd[k] - scp[k] * x;
        sd[k] = x;
        acc += x * sw[k];
    }
    sd[4 * nzp] = acc * a.inv_lz;
}
CANS_HD void z_singular_store(const ZArgs& a, const double* sd, int nzp, int tid, int nthreads) {
    const double mean = sd[4 * nzp];
    for (int k = tid; k < a.nz; k += nthreads) a.p[(size_t)k * a.ncols] = sd[k] - mean;
}

}  // namespace cans
