// chkdt_pass.cuh -- the stable-time-step reduction of Listing 1 (eq. 4):
//   dti = max_ijk max(dtix, dtiy, dtiz),   each the magnitude of the component living on that face times its inverse
//   spacing plus the 4-point face averages of the other two:
//   dtix = |u|/dx + |v(i,j)+v(i,j-1)+v(i+1,j)+v(i+1,j-1)|/(4 dy) + |w(i,j,k)+w(i,j,k-1)+w(i+1,j,k)+w(i+1,j,k-1)|/(4 dzf_k)
//   dtiy = |u(i,j)+u(i,j+1)+u(i-1,j+1)+u(i-1,j)|/(4 dx) + |v|/dy + |w(i,j,k)+w(i,j+1,k)+w(i,j+1,k-1)+w(i,j,k-1)|/(4 dzf_k)
//   dtiz = |u(i,j,k)+u(i-1,j,k)+u(i-1,j,k+1)+u(i,j,k+1)|/(4 dx) + |v(i,j,k)+v(i,j-1,k)+v(i,j-1,k+1)+v(i,j,k+1)|/(4 dy) + |w|/dzc_{k+1}
// on the compact halo-free layout.  Neighbours outside the arrays (reading S17): wrapped in a periodic direction;
// otherwise the layer below index 0 is the lower boundary face for the normal component (registered plane or 0) and 0 for
// a tangential one, the layer above the last index is 0.
//
// Mapping: as the correction kernel -- a thread owns a pair of x-adjacent cells of one row and marches up CHK_KC planes,
// carrying the rows of plane k+1 (u, v) and of plane k (w) into the next step, so every value comes from HBM once (the
// neighbour rows are other threads' own rows and come from L1 / L2): 24 B/cell.
#pragma once
#include "common.cuh"

namespace cans {

struct ChkArgs {
    int nx, ny, nz;
    const double* u; const double* v; const double* w;
    const double* fx; const double* fy; const double* fz;    // lower-face planes or NULL (as XYArgs)
    int wrap_x, wrap_y, wrap_z;
    double rdx, rdy;
    const double* rdzf;       // [nz] 1/dzf[k]
    const double* rdzc;       // [nz] 1/dzc[k+1]
    unsigned long long* dti;  // device scalar: bit pattern of a non-negative double, atomicMax'ed
};

struct Row3 { double a, b, c; };

#if defined(__CUDACC__)
// A row is fetched in two steps so that a thread has all its loads in flight before it consumes any of them (a warp
// issues in order: a shuffle right behind its load would serialise the loads).  Step 1 (chk_load_*): the pair (x0, x0+1)
// as one 16-byte load, plus -- only at a row end or a warp edge -- the outer value, loaded or synthesised by the boundary
// rule.  Step 2 (chk_left / chk_right): the outer value from the neighbouring lane's pair by shuffle (every lane of the
// warp takes part: cols is a multiple of 32), replaced by the edge value where step 1 fetched one.
struct RowLoad { double2 t; double edge; };

// u(i-1 | i, i+1) of row jj, plane kk
CANS_D RowLoad chk_load_u(const ChkArgs& a, int i, int jj, int kk, int lane) {
    bool in = true;
    if (jj >= a.ny) { in = a.wrap_y != 0; jj = 0; }
    if (kk >= a.nz) { in = in && a.wrap_z != 0; kk = 0; }
    const size_t ro = ((size_t)kk * a.ny + jj) * a.nx;
    RowLoad r;
    r.t = in ? *reinterpret_cast<const double2*>(a.u + ro + i) : make_double2(0.0, 0.0);
    r.edge = 0.0;
    if (in && (i == 0 || lane == 0)) {
        if (i > 0) r.edge = a.u[ro + i - 1];
        else if (a.wrap_x) r.edge = a.u[ro + a.nx - 1];
        else if (a.fx) r.edge = a.fx[(size_t)kk * a.ny + jj];
    }
    return r;
}
CANS_D Row3 chk_left(const RowLoad& l, int i, int lane) {
    double left = __shfl_up_sync(0xffffffffu, l.t.y, 1);
    if (i == 0 || lane == 0) left = l.edge;
    Row3 r = {left, l.t.x, l.t.y};
    return r;
}
// v or w (i, i+1 | i+2) of a row given by its base pointer (NULL: the row is outside and reads as 0)
CANS_D RowLoad chk_load_row(const double* row, int i, int nx, int wrap_x, int lane) {
    RowLoad r;
    r.t = row ? *reinterpret_cast<const double2*>(row + i) : make_double2(0.0, 0.0);
    r.edge = 0.0;
    if (row && (i + 2 >= nx || lane == 31)) {
        if (i + 2 < nx) r.edge = row[i + 2];
        else if (wrap_x) r.edge = row[0];
    }
    return r;
}
CANS_D Row3 chk_right(const RowLoad& l, int i, int nx, int lane) {
    double right = __shfl_down_sync(0xffffffffu, l.t.x, 1);
    if (i + 2 >= nx || lane == 31) right = l.edge;
    Row3 r = {l.t.x, l.t.y, right};
    return r;
}
// v(i, i+1 | i+2) of row jj (may be -1), plane kk
CANS_D RowLoad chk_load_v(const ChkArgs& a, int i, int jj, int kk, int lane) {
    const double* row = nullptr;
    bool in = true;
    if (kk >= a.nz) { in = a.wrap_z != 0; kk = 0; }
    if (in) {
        if (jj >= 0) row = a.v + ((size_t)kk * a.ny + jj) * a.nx;
        else if (a.wrap_y) row = a.v + ((size_t)kk * a.ny + a.ny - 1) * a.nx;
        else if (a.fy) row = a.fy + (size_t)kk * a.nx;
    }
    return chk_load_row(row, i, a.nx, a.wrap_x, lane);
}
// w(i, i+1 | i+2) of row jj (may be ny), plane kk (may be -1)
CANS_D RowLoad chk_load_w(const ChkArgs& a, int i, int jj, int kk, int lane) {
    const double* row = nullptr;
    bool in = true;
    if (jj >= a.ny) { in = a.wrap_y != 0; jj = 0; }
    if (in) {
        if (kk >= 0) row = a.w + ((size_t)kk * a.ny + jj) * a.nx;
        else if (a.wrap_z) row = a.w + ((size_t)(a.nz - 1) * a.ny + jj) * a.nx;
        else if (a.fz) row = a.fz + (size_t)jj * a.nx;
    }
    return chk_load_row(row, i, a.nx, a.wrap_x, lane);
}
// the six face sums of the pair of cells (i, i+1) of plane k from the eleven rows a thread holds; returns their maximum
CANS_D double chk_cell_max(const ChkArgs& a, int k, const Row3& uj, const Row3& up, const Row3& un, const Row3& vm,
                            const Row3& vj, const Row3& vmn, const Row3& vjn, const Row3& wlj, const Row3& wlp,
                            const Row3& wj, const Row3& wp) {
    const double qx = 0.25 * a.rdx, qy = 0.25 * a.rdy;
    const double rzf = a.rdzf[k], rzc = a.rdzc[k], qz = 0.25 * rzf;
    // cell i (values .a / .b of the v, w rows; .b of the u rows) and cell i+1 (.b / .c; .c)
    const double dtix0 = fabs(uj.b) * a.rdx + fabs(vj.a + vm.a + vj.b + vm.b) * qy + fabs(wj.a + wlj.a + wj.b + wlj.b) * qz;
    const double dtix1 = fabs(uj.c) * a.rdx + fabs(vj.b + vm.b + vj.c + vm.c) * qy + fabs(wj.b + wlj.b + wj.c + wlj.c) * qz;
    const double dtiy0 = fabs(uj.b + up.b + up.a + uj.a) * qx + fabs(vj.a) * a.rdy + fabs(wj.a + wp.a + wlp.a + wlj.a) * qz;
    const double dtiy1 = fabs(uj.c + up.c + up.b + uj.b) * qx + fabs(vj.b) * a.rdy + fabs(wj.b + wp.b + wlp.b + wlj.b) * qz;
    const double dtiz0 = fabs(uj.b + uj.a + un.a + un.b) * qx + fabs(vj.a + vm.a + vmn.a + vjn.a) * qy + fabs(wj.a) * rzc;
    const double dtiz1 = fabs(uj.c + uj.b + un.b + un.c) * qx + fabs(vj.b + vm.b + vmn.b + vjn.b) * qy + fabs(wj.b) * rzc;
    return fmax(fmax(dtix0, dtix1), fmax(fmax(dtiy0, dtiy1), fmax(dtiz0, dtiz1)));
}
#endif

}  // namespace cans
