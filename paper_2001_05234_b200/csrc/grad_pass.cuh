// grad_pass.cuh -- a7: velocity correction u -= dt G Phi (eq. 2c) on the compact staggered layout:
//   u_i -= dt (Phi_{i+1} - Phi_i)/dx,  v_j -= dt (Phi_{j+1} - Phi_j)/dy,  w_k -= dt (Phi_{k+1} - Phi_k)/dzc_{k+1};
// Phi beyond the upper face follows the ghost rule (P wrap, N mirror, D anti-mirror), so the value on an
// upper 'N' face is left bit-identical.
#pragma once
#include "common.cuh"

namespace cans {

struct GradArgs {
    int nx, ny, nz;
    double* u; double* v; double* w;
    const double* phi;
    const double* rdzc;        // [nz] 1/dzc[k+1]
    double dt_rdx, dt_rdy, dt;
    // ghost rule beyond the upper face: value = sgn * phi[idx]  (P: idx 0, sgn 1; N: idx n-1, sgn 1; D: idx n-1, sgn -1)
    int gx_idx, gy_idx, gz_idx;
    double gx_sgn, gy_sgn, gz_sgn;
};

// one pair of x-adjacent cells (t = pair index, x fastest)
CANS_HD void grad_correct_pair(const GradArgs& a, size_t t) {
    const size_t plane = (size_t)a.nx * a.ny;
    const int hx = a.nx / 2;
    const int i = 2 * (int)(t % hx);
    const size_t row = t / hx;
    const int j = (int)(row % a.ny);
    const int k = (int)(row / a.ny);
    const size_t o = (size_t)k * plane + (size_t)j * a.nx + i;
    const double2 ph = *reinterpret_cast<const double2*>(a.phi + o);
    // x neighbour of the second cell
    double phx = (i + 2 < a.nx) ? a.phi[o + 2] : a.gx_sgn * a.phi[o - i + a.gx_idx];
    // y neighbours
    double2 phy;
    if (j + 1 < a.ny) phy = *reinterpret_cast<const double2*>(a.phi + o + a.nx);
    else {
        phy = *reinterpret_cast<const double2*>(a.phi + (size_t)k * plane + (size_t)a.gy_idx * a.nx + i);
        phy.x *= a.gy_sgn; phy.y *= a.gy_sgn;
    }
    double2 phz;
    if (k + 1 < a.nz) phz = *reinterpret_cast<const double2*>(a.phi + o + plane);
    else {
        phz = *reinterpret_cast<const double2*>(a.phi + (size_t)a.gz_idx * plane + (size_t)j * a.nx + i);
        phz.x *= a.gz_sgn; phz.y *= a.gz_sgn;
    }
    double2 uu = *reinterpret_cast<double2*>(a.u + o);
    double2 vv = *reinterpret_cast<double2*>(a.v + o);
    double2 ww = *reinterpret_cast<double2*>(a.w + o);
    uu.x -= a.dt_rdx * (ph.y - ph.x);
    uu.y -= a.dt_rdx * (phx - ph.y);
    vv.x -= a.dt_rdy * (phy.x - ph.x);
    vv.y -= a.dt_rdy * (phy.y - ph.y);
    const double dz = a.dt * a.rdzc[k];
    ww.x -= dz * (phz.x - ph.x);
    ww.y -= dz * (phz.y - ph.y);
    *reinterpret_cast<double2*>(a.u + o) = uu;
    *reinterpret_cast<double2*>(a.v + o) = vv;
    *reinterpret_cast<double2*>(a.w + o) = ww;
}

}  // namespace cans
