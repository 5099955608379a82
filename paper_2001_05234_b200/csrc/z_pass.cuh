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
//     accumulating the propagation factor (prod of -a_k r_k, resp. -c_k r_k); a P-step scan over the
//     segment ends in shared memory supplies the true start value, which is then propagated;
//   * results go straight from registers to global memory (coalesced rows).
// The singular kx = ky = 0 column of an all-periodic/Neumann problem is handled by z_singular_column
// (CTA 0, before it joins the tile loop).
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
    int nbox, box_rows;       // TMA tiling of a column tile: nbox boxes of box_rows rows (set by z_solve_launch)
};

// one pivot step; shared by the plan-time table kernel and the solve so the values are identical
// The reciprocal is the hardware seed (rcp.approx, ~20 bits) refined by two Newton steps: full double precision
// to about one unit in the last place for these well-scaled, strictly negative denominators, without the range
// checks and the slow path of the IEEE division -- the pivot chain is the longest dependency chain of the solve.
CANS_HD double z_pivot(double bk, double lam, double gk, double rprev) {
    const double den = (bk + lam) - gk * rprev;
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

template <int MROWS>
struct ZState {
    double d[MROWS];
    double r[MROWS];
    double start;     // true d'_{k0-1}, later true x_{k0+MROWS}
    long col;
    bool active;
};

// shared memory (doubles): tables az,bz,cz,gz [4][nzp]; scan arrays end[TC*P], fac[TC*P] of the forward sweep and a
// second pair for the backward sweep (so that no barrier is needed between reading one and writing the other);
// two tile buffers [nzp][TC]
template <int MROWS, int TC>
struct ZPass {
    static CANS_HD size_t table_doubles(int nseg) { return (size_t)4 * nseg * MROWS + (size_t)4 * TC * nseg; }
    static CANS_HD size_t tile_doubles(int nseg) { return (size_t)nseg * MROWS * TC; }
    static CANS_HD size_t smem_doubles(int nseg) { return table_doubles(nseg) + 2 * tile_doubles(nseg); }

    static CANS_HD void load_tables(const ZArgs& a, double* sm, int tid, int nthreads) {
        const int nzp = a.nseg * MROWS;
        for (int i = tid; i < nzp; i += nthreads) {
            sm[i] = a.az[i];
            sm[nzp + i] = a.bz[i];
            sm[2 * nzp + i] = a.cz[i];
            sm[3 * nzp + i] = a.gz[i];
        }
    }

    // phase 1: take the segment from the tile buffer, pivots, local forward sweep from a zero start;
    // publish (end, factor)
    static CANS_HD void phase1(const ZArgs& a, double* sm, const double* buf, ZState<MROWS>& st, long tile,
                               double rstart_val, double lam, int tid) {
        const int nzp = a.nseg * MROWS;
        const double* saz = sm;
        const double* sbz = sm + nzp;
        const double* sgz = sm + 3 * nzp;
        double2* s_scan = reinterpret_cast<double2*>(sm + 4 * nzp);      // forward (end, factor) pairs
        const int c = tid % TC;
        const int s = tid / TC;
        const long col = tile * TC + c;
        st.col = col;
        st.active = (col < a.ncols) && !(a.singular && col == 0);
        const int k0 = s * MROWS;
        if (col < a.ncols) {
#pragma unroll
            for (int r = 0; r < MROWS; ++r) {
                const int k = k0 + r;
                st.d[r] = (k < a.nz) ? buf[(size_t)k * TC + c] * a.scale : 0.0;
            }
            double rp = rstart_val;
            double dp = 0.0, fac = 1.0;
#pragma unroll
            for (int r = 0; r < MROWS; ++r) {
                const int k = k0 + r;
                rp = z_pivot(sbz[k], lam, sgz[k], rp);
                st.r[r] = rp;
                const double e = saz[k] * rp;
                dp = st.d[r] * rp - e * dp;
                st.d[r] = dp;
                fac *= -e;
            }
            s_scan[s * TC + c] = make_double2(dp, fac);
        } else {
            s_scan[s * TC + c] = make_double2(0.0, 0.0);
        }
    }

    // phase 2: scan the segment ends -> true start; propagate; local backward sweep from a zero start; publish
    static CANS_HD void phase2a(const ZArgs& a, double* sm, ZState<MROWS>& st, int tid) {
        const int nzp = a.nseg * MROWS;
        const double2* s_scan = reinterpret_cast<const double2*>(sm + 4 * nzp);
        const int c = tid % TC;
        const int s = tid / TC;
        double D = 0.0;                     // true d' at the end of segment s'-1
#pragma unroll 4
        for (int q = 0; q < s; ++q) {
            const double2 ef = s_scan[q * TC + c];      // one 16-byte load per segment
            D = ef.x + ef.y * D;
        }
        st.start = D;
    }
    // (2b publishes into the backward pair of scan arrays, so 2a and 2b need no barrier between them)
    static CANS_HD void phase2b(const ZArgs& a, double* sm, ZState<MROWS>& st, int tid) {
        const int nzp = a.nseg * MROWS;
        const double* saz = sm;
        const double* scz = sm + 2 * nzp;
        double2* s_scan = reinterpret_cast<double2*>(sm + 4 * nzp + 2 * TC * a.nseg);   // backward pairs
        const int c = tid % TC;
        const int s = tid / TC;
        const int k0 = s * MROWS;
        if (st.col < a.ncols) {
            double fac = 1.0;
            const double D = st.start;
#pragma unroll
            for (int r = 0; r < MROWS; ++r) {
                fac *= -(saz[k0 + r] * st.r[r]);
                st.d[r] += fac * D;
            }
            double xs = 0.0, g = 1.0;
#pragma unroll
            for (int r = MROWS - 1; r >= 0; --r) {
                const double cp = scz[k0 + r] * st.r[r];
                xs = st.d[r] - cp * xs;
                st.d[r] = xs;
                g *= -cp;
            }
            s_scan[s * TC + c] = make_double2(xs, g);     // x^0 at the top row of the segment, its factor
        } else {
            s_scan[s * TC + c] = make_double2(0.0, 0.0);
        }
    }

    // phase 3: scan from the bottom -> true x below the segment; propagate; store
    static CANS_HD void phase3(const ZArgs& a, double* sm, ZState<MROWS>& st, int tid) {
        const int nzp = a.nseg * MROWS;
        const double* scz = sm + 2 * nzp;
        const double2* s_scan = reinterpret_cast<const double2*>(sm + 4 * nzp + 2 * TC * a.nseg);   // backward pairs
        const int c = tid % TC;
        const int s = tid / TC;
        const int k0 = s * MROWS;
        double X = 0.0;                     // true x at the top row of segment s'+1
#pragma unroll 4
        for (int q = a.nseg - 1; q > s; --q) {
            const double2 ef = s_scan[q * TC + c];
            X = ef.x + ef.y * X;
        }
        if (st.active) {
            const size_t plane = (size_t)a.ncols;
            double g = 1.0;
#pragma unroll
            for (int r = MROWS - 1; r >= 0; --r) {
                g *= -(scz[k0 + r] * st.r[r]);
                st.d[r] += g * X;
            }
#pragma unroll
            for (int r = 0; r < MROWS; ++r) {
                const int k = k0 + r;
                if (k < a.nz) a.p[(size_t)k * plane + st.col] = st.d[r];
            }
        }
    }
};

// plan-time: pivots at the segment boundaries of every column (thread per column, sequential in k)
template <int MROWS>
CANS_HD void z_setup_column(const ZArgs& a, double* rstart_out, double* r00_out, long col) {
    const int i = (int)(col % a.nx);
    const int j = (int)(col / a.nx);
    const double lam = a.lamx[i] + a.lamy[j];
    double rp = 0.0;
    const int nzp = a.nseg * MROWS;
    for (int k = 0; k < nzp; ++k) {
        if (k % MROWS == 0) rstart_out[(size_t)(k / MROWS) * a.ncols + col] = rp;
        rp = z_pivot(a.bz[k], lam, a.gz[k], rp);
        if (col == 0 && k < a.nz && r00_out) r00_out[k] = rp;
    }
}

// The singular column (reading S3 / oracle O4): forward sweep on rows 0..nz-2, x[nz-1] = 0,
// back-substitute, subtract the dzf-weighted mean.  One thread; d is staged in shared memory.
CANS_HD void z_singular_column(const ZArgs& a, double* sd /* nz doubles */) {
    const size_t plane = (size_t)a.ncols;
    const int nz = a.nz;
    double dp = 0.0;
    for (int k = 0; k < nz - 1; ++k) {
        const double rk = a.r00[k];
        dp = (sd[k] * a.scale - a.az[k] * dp) * rk;
        sd[k] = dp;
    }
    double x = 0.0, acc = 0.0;
    sd[nz - 1] = 0.0;
    for (int k = nz - 2; k >= 0; --k) {
        x = sd[k] - a.cz[k] * a.r00[k] * x;
        sd[k] = x;
        acc += x * a.dzf[k];
    }
    const double mean = acc * a.inv_lz;
    for (int k = 0; k < nz; ++k) a.p[(size_t)k * plane] = sd[k] - mean;
}

}  // namespace cans
