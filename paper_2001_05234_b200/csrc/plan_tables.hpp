// plan_tables.hpp -- host-side tables of a plan: eigenvalues per spectral position, twiddles,
// z-operator rows.  Plain C++ (no CUDA), written for the layouts of xy_pass.cuh / z_pass.cuh.
//
//   lam per position: eigenvalue of the undivided 1-D second difference (eq. 6 lambda_i, lambda_j,
//                     P:L102) of the mode stored at that slot position (see xy_pass.cuh header).
//   z rows:           a_k = 1/(dzf_k dzc_k), c_k = 1/(dzf_k dzc_{k+1}), b_k = -(a_k + c_k) with the
//                     boundary rows folded in (ghost = +interior for 'N', -interior for 'D').
#pragma once
#include <cmath>
#include <cstddef>
#include <vector>

#include "fft_sizes.h"

namespace cans {

struct FftRadices { int n, r1, r2, r3, nfx, ntx, txc, nty; };

inline bool fft_lookup(int n, FftRadices* out) {
#define CANS_ROW(N, R1, R2, R3, NFX, NTX, TXC, NTY) \
    if (n == N) { *out = FftRadices{N, R1, R2, R3, NFX, NTX, TXC, NTY}; return true; }
    CANS_FFT_SIZES(CANS_ROW)
#undef CANS_ROW
    return false;
}

// exp(-2 pi i num / den), argument reduced exactly in integers to the first octant, long double trig
inline void unit_root(long long num, long long den, double* re, double* im) {
    num %= den;
    if (num < 0) num += den;
    // angle = 2 pi num/den in [0, 2 pi); work with eighths of a turn: t = 8 num / den
    const long double PI = 3.14159265358979323846264338327950288L;
    long long oct = (8 * num) / den;            // 0..7
    long long rem = 8 * num - oct * den;        // remainder, angle within the octant = (pi/4) rem/den
    long double c, s;
    if ((oct & 1) == 0) {
        long double th = (PI / 4) * (long double)rem / (long double)den;
        c = cosl(th); s = sinl(th);
    } else {
        long double th = (PI / 4) * (long double)(den - rem) / (long double)den;
        c = sinl(th); s = cosl(th);             // cos(pi/4 + x) with x -> pi/4 - th reflection
    }
    // (c, s) now are cos/sin of the angle folded into [0, pi/2) pieces: oct even: angle_in_quadrant = th (<pi/4),
    // oct odd: angle_in_quadrant = pi/2 - th'.  Rotate by quadrant = oct / 2.
    long double cq, sq;
    cq = c; sq = s;
    long double cr, sr;
    switch (oct / 2) {
        case 0: cr = cq; sr = sq; break;
        case 1: cr = -sq; sr = cq; break;
        case 2: cr = -cq; sr = -sq; break;
        default: cr = sq; sr = -cq; break;
    }
    *re = (double)cr;
    *im = (double)(-sr);
}

// pass twiddle table of FftPlan (fft_core.cuh): pass 1 [k-1][p] = W_N^(p k), pass 2 [k-1][p] = W_(N/R1)^(p k)
inline std::vector<double> make_pass_twiddles(const FftRadices& f) {
    const int s1 = f.r2 * f.r3, s2 = f.r3, m2 = f.n / f.r1;
    std::vector<double> t;
    for (int k = 1; k < f.r1; ++k)
        for (int p = 0; p < s1; ++p) {
            double re, im;
            unit_root((long long)p * k, f.n, &re, &im);
            t.push_back(re); t.push_back(im);
        }
    if (f.r2 > 1)
        for (int k = 1; k < f.r2; ++k)
            for (int p = 0; p < s2; ++p) {
                double re, im;
                unit_root((long long)p * k, m2, &re, &im);
                t.push_back(re); t.push_back(im);
            }
    return t;
}

// twiddles between the two passes of the warp-per-line transform (xw_pass.cuh): [k1][p] = W_n^(p k1), p < 32, k1 < n/32
inline std::vector<double> make_two_pass_twiddles(int n) {
    std::vector<double> t;
    for (int k1 = 0; k1 < n / 32; ++k1)
        for (int p = 0; p < 32; ++p) {
            double re, im;
            unit_root((long long)p * k1, n, &re, &im);
            t.push_back(re); t.push_back(im);
        }
    return t;
}

// w^q = exp(-i pi q / (2n)) = exp(-2 pi i q / (4n)), q = 0..n/2-1
inline std::vector<double> make_post_twiddles(int n) {
    std::vector<double> t;
    for (int q = 0; q < n / 2; ++q) {
        double re, im;
        unit_root(q, 4LL * n, &re, &im);
        t.push_back(re); t.push_back(im);
    }
    return t;
}

// mixed pairs (DCT-IV / DST-IV): post-twiddles exp(-i pi (2q+1) / (4n)), q = 0..n/2-1 ...
inline std::vector<double> make_post_twiddles_mixed(int n) {
    std::vector<double> t;
    for (int q = 0; q < n / 2; ++q) {
        double re, im;
        unit_root(2 * q + 1, 8LL * n, &re, &im);
        t.push_back(re); t.push_back(im);
    }
    return t;
}
// ... and pre-twiddles exp(-i pi m / n), m = 0..n-1
inline std::vector<double> make_pre_twiddles_mixed(int n) {
    std::vector<double> t;
    for (int m = 0; m < n; ++m) {
        double re, im;
        unit_root(m, 2LL * n, &re, &im);
        t.push_back(re); t.push_back(im);
    }
    return t;
}

// -4 sin^2(pi num / den)
inline double lam_sin2(long long num, long long den) {
    double re, im;
    unit_root(num, 2 * den, &re, &im);     // exp(-i pi num/den): im = -sin(pi num/den)
    return -4.0 * im * im;
}

// eigenvalue of the mode stored at every slot position of a line of n (kind: 0 PP, 1 NN, 2 DD, 3 ND, 4 DN), divided by h^2
inline std::vector<double> make_lambda_positions(int n, int kind, double h) {
    std::vector<double> lam(n);
    const double ih2 = 1.0 / (h * h);
    if (kind >= 3) {
        // mixed pairs: mode q has -4 sin^2(pi (2q+1) / (4n)); positions (2s, 2s+1) hold modes (s, n-1-s) for ND, (n-1-s, s) for DN
        for (int s = 0; s < n / 2; ++s) {
            const double lo = lam_sin2(2LL * s + 1, 4LL * n) * ih2, hi = lam_sin2(2LL * (n - 1 - s) + 1, 4LL * n) * ih2;
            lam[2 * s] = (kind == 3) ? lo : hi;
            lam[2 * s + 1] = (kind == 3) ? hi : lo;
        }
        return lam;
    }
    auto mode = [&](int q) -> double {
        if (kind == 0) return lam_sin2(q, n);                 // PP: frequency q
        if (kind == 1) return lam_sin2(q, 2LL * n);           // NN: cosine mode q
        return lam_sin2(n - q, 2LL * n);                      // DD: slot of C'_q holds sine mode n-1-q
    };
    lam[0] = mode(0) * ih2;
    lam[1] = mode(n / 2) * ih2;
    for (int q = 1; q < n / 2; ++q) {
        lam[2 * q] = mode(q) * ih2;
        lam[2 * q + 1] = ((kind == 0) ? mode(q) : mode(n - q)) * ih2;
    }
    return lam;
}

struct ZRows {
    std::vector<double> a, b, c, g, rdzf, dzf;   // a,b,c,g padded to nzp; rdzf, dzf of length nz
    double lz_sum;
    double a0w, cw;                              // a_0 and c_{nz-1} before they were zeroed
};

// lo / up: 'N' or 'D', or both 'P' (cyclic system: no boundary folding, the wrap couplings a_0 and c_{nz-1} are returned
// separately and zeroed in the rows).  nzp >= nz: rows beyond nz are decoupled identity-like rows (a = c = g = 0, b = -1).
// face != 0: the unknown lives on the +z faces (wall-normal velocity of eq. 3b): a_k = 1/(dzc_{k+1} dzf_k),
// c_k = 1/(dzc_{k+1} dzf_{k+1}); walls ('D','D'): rows 0..nz-2, wall nodes carry no coupling; periodic: wrapped;
// wall below and zero slope at the top ('D','N'): rows 0..nz-1, the last with a mirrored upper neighbour.
inline ZRows make_z_rows(int nz, int nzp, const double* dzc, const double* dzf, char lo, char up, int face = 0) {
    ZRows z;
    if (face) {
        z.a.assign(nzp, 0.0); z.b.assign(nzp, -1.0); z.c.assign(nzp, 0.0); z.g.assign(nzp, 0.0);
        z.rdzf.resize(nz); z.dzf.resize(nz);
        z.lz_sum = 0.0;
        const bool open_top = (lo == 'D' && up == 'N');      // zero slope AT the upper boundary face: face nz-1 is an unknown
        const int rows = (lo == 'P' || open_top) ? nz : nz - 1;
        for (int k = 0; k < nz; ++k) { z.rdzf[k] = 1.0 / dzf[k]; z.dzf[k] = dzf[k]; z.lz_sum += dzf[k]; }
        for (int k = 0; k < rows; ++k) {
            z.a[k] = 1.0 / (dzc[k + 1] * dzf[k]);
            z.c[k] = 1.0 / (dzc[k + 1] * dzf[(k + 1) % nz]);
            z.b[k] = -(z.a[k] + z.c[k]);
        }
        if (open_top) {
            // the face above face nz-1 is the mirror image of face nz-2 (ghost cell of width dzf_{nz-1}): its coupling
            // folds into a_{nz-1}
            const double ghost = 1.0 / (dzc[nz] * dzf[nz - 1]);
            z.b[nz - 1] = -(z.a[nz - 1] + ghost);
            z.a[nz - 1] += ghost;
            z.c[nz - 1] = 0.0;
        }
        z.a0w = z.a[0];
        z.cw = z.c[rows - 1];
        z.a[0] = 0.0;
        z.c[rows - 1] = 0.0;
        for (int k = 1; k < rows; ++k) z.g[k] = z.a[k] * z.c[k - 1];
        return z;
    }
    z.a.assign(nzp, 0.0); z.b.assign(nzp, -1.0); z.c.assign(nzp, 0.0); z.g.assign(nzp, 0.0);
    z.rdzf.resize(nz); z.dzf.resize(nz);
    z.lz_sum = 0.0;
    for (int k = 0; k < nz; ++k) {
        const double ak = 1.0 / (dzf[k] * dzc[k]);
        const double ck = 1.0 / (dzf[k] * dzc[k + 1]);
        z.a[k] = ak; z.c[k] = ck; z.b[k] = -(ak + ck);
        z.rdzf[k] = 1.0 / dzf[k];
        z.dzf[k] = dzf[k];
        z.lz_sum += dzf[k];
    }
    z.a0w = z.a[0];
    z.cw = z.c[nz - 1];
    if (lo != 'P') {
        z.b[0] += (lo == 'N') ? z.a[0] : -z.a[0];
        z.b[nz - 1] += (up == 'N') ? z.c[nz - 1] : -z.c[nz - 1];
    }
    z.a[0] = 0.0;
    z.c[nz - 1] = 0.0;
    for (int k = 1; k < nz; ++k) z.g[k] = z.a[k] * z.c[k - 1];
    return z;
}

}  // namespace cans
