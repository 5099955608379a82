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
// u(i-1, i, i+1) of row jj, plane kk (i even, i+1 < nx)
CANS_D Row3 chk_row_u(const ChkArgs& a, int i, int jj, int kk) {
    Row3 r = {0.0, 0.0, 0.0};
    if (jj >= a.ny) { if (!a.wrap_y) return r; jj = 0; }
    if (kk >= a.nz) { if (!a.wrap_z) return r; kk = 0; }
    const size_t ro = ((size_t)kk * a.ny + jj) * a.nx;
    const double2 t = *reinterpret_cast<const double2*>(a.u + ro + i);
    r.b = t.x; r.c = t.y;
    if (i > 0) r.a = a.u[ro + i - 1];
    else if (a.wrap_x) r.a = a.u[ro + a.nx - 1];
    else if (a.fx) r.a = a.fx[(size_t)kk * a.ny + jj];
    return r;
}
// v(i, i+1, i+2) of row jj (may be -1), plane kk
CANS_D Row3 chk_row_v(const ChkArgs& a, int i, int jj, int kk) {
    Row3 r = {0.0, 0.0, 0.0};
    if (kk >= a.nz) { if (!a.wrap_z) return r; kk = 0; }
    const double* row;
    if (jj >= 0) row = a.v + ((size_t)kk * a.ny + jj) * a.nx;
    else if (a.wrap_y) row = a.v + ((size_t)kk * a.ny + a.ny - 1) * a.nx;
    else if (a.fy) row = a.fy + (size_t)kk * a.nx;
    else return r;
    const double2 t = *reinterpret_cast<const double2*>(row + i);
    r.a = t.x; r.b = t.y;
    if (i + 2 < a.nx) r.c = row[i + 2];
    else if (a.wrap_x) r.c = row[0];
    return r;
}
// w(i, i+1, i+2) of row jj (may be ny), plane kk (may be -1)
CANS_D Row3 chk_row_w(const ChkArgs& a, int i, int jj, int kk) {
    Row3 r = {0.0, 0.0, 0.0};
    if (jj >= a.ny) { if (!a.wrap_y) return r; jj = 0; }
    const double* row;
    if (kk >= 0) row = a.w + ((size_t)kk * a.ny + jj) * a.nx;
    else if (a.wrap_z) row = a.w + ((size_t)(a.nz - 1) * a.ny + jj) * a.nx;
    else if (a.fz) row = a.fz + (size_t)jj * a.nx;
    else return r;
    const double2 t = *reinterpret_cast<const double2*>(row + i);
    r.a = t.x; r.b = t.y;
    if (i + 2 < a.nx) r.c = row[i + 2];
    else if (a.wrap_x) r.c = row[0];
    return r;
}
#endif

}  // namespace cans
