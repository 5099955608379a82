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
    // eq. 3e, LAP instantiation only: pacc += Phi - lap_coef * L Phi with the 7-point Laplacian of eq. 5 taken from
    // the values the thread already holds plus Phi(i-1), Phi(j-1) (cache hits: the neighbouring threads' own values) and
    // the plane below, which it carries.  Ghost rule below the lower face, as above: value = sgn * phi[idx]
    // (P: idx n-1, sgn 1; N: idx 0, sgn 1; D: idx 0, sgn -1).
    double lap_coef, rdx2, rdy2, rdzc0;   // gamma nu dt / 2;  1/dx^2, 1/dy^2;  1/dzc[0]
    const double* rdzf;                   // [nz] 1/dzf[k]
    int lx_idx, ly_idx, lz_idx;
    double lx_sgn, ly_sgn, lz_sgn;
};

// inputs of one pair of x-adjacent cells, fetched before any of them is used
struct GradIn {
    double2 ph, phy, phz, uu, vv, ww, pa;
    double2 phym, phzm;        // LAP only: row j-1 and plane k-1 (ghost rule applied)
    double phx, phxm;          // Phi(i+2); LAP only: Phi(i-1)
    size_t o;
    int k;
};

template <bool LAP = false>
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
    if (LAP) {
        const double rf = a.rdzf[in.k];
        const double az = rf * (in.k > 0 ? a.rdzc[in.k - 1] : a.rdzc0), cz = rf * a.rdzc[in.k];   // a_k, c_k of the z operator
        const double lx0 = (in.phxm - 2.0 * ph.x + ph.y) * a.rdx2 + (in.phym.x - 2.0 * ph.x + in.phy.x) * a.rdy2 +
                           az * (in.phzm.x - ph.x) + cz * (in.phz.x - ph.x);
        const double lx1 = (ph.x - 2.0 * ph.y + in.phx) * a.rdx2 + (in.phym.y - 2.0 * ph.y + in.phy.y) * a.rdy2 +
                           az * (in.phzm.y - ph.y) + cz * (in.phz.y - ph.y);
        *reinterpret_cast<double2*>(a.pacc + in.o) =
            make_double2(in.pa.x + ph.x - a.lap_coef * lx0, in.pa.y + ph.y - a.lap_coef * lx1);
    } else if (a.pacc) {
        *reinterpret_cast<double2*>(a.pacc + in.o) = make_double2(in.pa.x + ph.x, in.pa.y + ph.y);
    }
}

}  // namespace cans
