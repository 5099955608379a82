// grad_pass.cuh -- a7: velocity correction u -= dt G Phi (eq. 2c) on the compact staggered layout:
//   u_i -= dt (Phi_{i+1} - Phi_i)/dx,  v_j -= dt (Phi_{j+1} - Phi_j)/dy,  w_k -= dt (Phi_{k+1} - Phi_k)/dzc_{k+1};
// Phi beyond the upper face follows the ghost rule (P wrap, N mirror, D anti-mirror), so the value on an
// upper 'N' face is left bit-identical.
#pragma once
#include "common.cuh"

namespace cans {

struct GradArgs {
    int nx, ny, nz;
    int k0, k1;                // planes [k0, k1) corrected by this launch
    double* u; double* v; double* w;
    const double* phi;
    double* pacc;              // eq. 2d: pacc += Phi in the same pass, or NULL
    const double* rdzc;        // [nz] 1/dzc[k+1]
    double dt_rdx, dt_rdy, dt;
    // ghost rule beyond the upper face: value = sgn * phi[idx]  (P: idx 0, sgn 1; N: idx n-1, sgn 1; D: idx n-1, sgn -1)
    int gx_idx, gy_idx, gz_idx;
    double gx_sgn, gy_sgn, gz_sgn;
};

// inputs of one pair of x-adjacent cells, fetched before any of them is used
struct GradIn {
    double2 ph, phy, phz, uu, vv, ww, pa;
    double phx;
    size_t o;
    int k;
};

CANS_HD void grad_apply(const GradArgs& a, const GradIn& in) {
    double2 uu = in.uu, vv = in.vv, ww = in.ww;
    const double2 ph = in.ph;
    uu.x -= a.dt_rdx * (ph.y - ph.x);
    uu.y -= a.dt_rdx * (in.phx - ph.y);
    vv.x -= a.dt_rdy * (in.phy.x - ph.x);
    vv.y -= a.dt_rdy * (in.phy.y - ph.y);
    const double dz = a.dt * a.rdzc[in.k];
    ww.x -= dz * (in.phz.x - ph.x);
    ww.y -= dz * (in.phz.y - ph.y);
    *reinterpret_cast<double2*>(a.u + in.o) = uu;
    *reinterpret_cast<double2*>(a.v + in.o) = vv;
    *reinterpret_cast<double2*>(a.w + in.o) = ww;
    if (a.pacc) *reinterpret_cast<double2*>(a.pacc + in.o) = make_double2(in.pa.x + ph.x, in.pa.y + ph.y);
}

}  // namespace cans
