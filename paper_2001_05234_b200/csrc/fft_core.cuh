// fft_core.cuh -- in-register complex DFT butterflies (radix 2,3,4,6,8,12,16) and the in-place
// shared-memory mixed-radix passes built on them.
//
// Forward  = decimation in frequency: natural-order input, digit-reversed output.
// Inverse  = the exact transpose (decimation in time): digit-reversed input, natural-order output,
//            unnormalised.  With N = R1*R2*R3 the frequency q = b + R1*b2 + R1*R2*b3 of a forward
//            transform ends up at location b*(R2*R3) + b2*R3 + b3   (digit_reversed_loc below).
//
// These are the x / y real-to-real transforms F^x, F^y of eq. 6 after the
// "two real lines -> one complex line" packing described in xy_pass.cuh.
#pragma once
#include "common.cuh"

namespace cans {

// cos(2 pi m / D), sin(2 pi m / D) for the two denominators the composite butterflies need.
template <int D> CANS_HD double tab_cos(int m);
template <> CANS_HD double tab_cos<16>(int m) {
    const double C1 = 0.92387953251128673848, C2 = 0.70710678118654752440, S1 = 0.38268343236508977173;
    switch (m & 15) {
        case 0: return 1.0;  case 1: return C1;   case 2: return C2;   case 3: return S1;
        case 4: return 0.0;  case 5: return -S1;  case 6: return -C2;  case 7: return -C1;
        case 8: return -1.0; case 9: return -C1;  case 10: return -C2; case 11: return -S1;
        case 12: return 0.0; case 13: return S1;  case 14: return C2;  default: return C1;
    }
}
template <> CANS_HD double tab_cos<12>(int m) {
    const double H = 0.86602540378443864676;
    m = ((m % 12) + 12) % 12;
    switch (m) {
        case 0: return 1.0;   case 1: return H;     case 2: return 0.5;  case 3: return 0.0;
        case 4: return -0.5;  case 5: return -H;    case 6: return -1.0; case 7: return -H;
        case 8: return -0.5;  case 9: return 0.0;   case 10: return 0.5; default: return H;
    }
}
template <int D> CANS_HD double tab_sin(int m) { return tab_cos<D>(m - D / 4); }

// v *= W_D^m   (forward: W = exp(-2 pi i / D); INV: conjugate), m a compile-time constant after unrolling
template <int D, bool INV>
CANS_HD cplx mul_root(cplx v, int m) {
    m = ((m % D) + D) % D;
    if (m == 0) return v;
    if (m == D / 2) return cneg(v);
    if (m == D / 4) return INV ? cmul_pi(v) : cmul_mi(v);
    if (m == 3 * D / 4) return INV ? cmul_mi(v) : cmul_pi(v);
    const double c = tab_cos<D>(m);
    const double s = INV ? tab_sin<D>(m) : -tab_sin<D>(m);
    return make_double2(v.x * c - v.y * s, v.x * s + v.y * c);
}

template <int R, bool INV> struct Dft;

template <bool INV> struct Dft<1, INV> {
    static CANS_HD void run(cplx (&)[1]) {}
};

template <bool INV> struct Dft<2, INV> {
    static CANS_HD void run(cplx (&v)[2]) {
        cplx a = v[0], b = v[1];
        v[0] = cadd(a, b);
        v[1] = csub(a, b);
    }
};

template <bool INV> struct Dft<3, INV> {
    static CANS_HD void run(cplx (&v)[3]) {
        const double H = 0.86602540378443864676;
        cplx s = cadd(v[1], v[2]);
        cplx d = cscale(csub(v[1], v[2]), H);
        cplx t = make_double2(v[0].x - 0.5 * s.x, v[0].y - 0.5 * s.y);
        cplx r = INV ? cmul_pi(d) : cmul_mi(d);       // -+ i * (sqrt3/2) (v1 - v2)
        v[0] = cadd(v[0], s);
        v[1] = cadd(t, r);
        v[2] = csub(t, r);
    }
};

template <bool INV> struct Dft<4, INV> {
    static CANS_HD void run(cplx (&v)[4]) {
        cplx t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]);
        cplx t2 = cadd(v[1], v[3]);
        cplx t3 = INV ? cmul_pi(csub(v[1], v[3])) : cmul_mi(csub(v[1], v[3]));
        v[0] = cadd(t0, t2);
        v[1] = cadd(t1, t3);
        v[2] = csub(t0, t2);
        v[3] = csub(t1, t3);
    }
};

// R = RA*RB: DFT_RA over a1 (stride RB), internal twiddle W_R^(a0*k1), DFT_RB over a0; output k = k1 + RA*k0.
template <int RA, int RB, int D, bool INV>
struct DftComposite {
    static constexpr int R = RA * RB;
    static CANS_HD void run(cplx (&v)[R]) {
        cplx u[RA][RB];
#pragma unroll
        for (int a0 = 0; a0 < RB; ++a0) {
            cplx t[RA];
#pragma unroll
            for (int a1 = 0; a1 < RA; ++a1) t[a1] = v[a1 * RB + a0];
            Dft<RA, INV>::run(t);
#pragma unroll
            for (int k1 = 0; k1 < RA; ++k1) u[k1][a0] = mul_root<D, INV>(t[k1], a0 * k1 * (D / R));
        }
#pragma unroll
        for (int k1 = 0; k1 < RA; ++k1) {
            Dft<RB, INV>::run(u[k1]);
#pragma unroll
            for (int k0 = 0; k0 < RB; ++k0) v[k1 + RA * k0] = u[k1][k0];
        }
    }
};

template <bool INV> struct Dft<8, INV> { static CANS_HD void run(cplx (&v)[8]) { DftComposite<2, 4, 16, INV>::run(v); } };
template <bool INV> struct Dft<16, INV> { static CANS_HD void run(cplx (&v)[16]) { DftComposite<4, 4, 16, INV>::run(v); } };
template <bool INV> struct Dft<6, INV> { static CANS_HD void run(cplx (&v)[6]) { DftComposite<3, 2, 12, INV>::run(v); } };
template <bool INV> struct Dft<12, INV> { static CANS_HD void run(cplx (&v)[12]) { DftComposite<3, 4, 12, INV>::run(v); } };

// ------------------------------------------------------------------------------------------------
// Compile-time plan of one transform length.
// ------------------------------------------------------------------------------------------------
template <int N_, int R1_, int R2_, int R3_>
struct FftPlan {
    static constexpr int N = N_, R1 = R1_, R2 = R2_, R3 = R3_;
    static_assert(R1_ * R2_ * R3_ == N_, "radices must multiply to N");
    static constexpr int S1 = R2 * R3;      // stride of pass 1
    static constexpr int M2 = S1;           // sub-transform length of pass 2
    static constexpr int S2 = R3;           // stride of pass 2
    // twiddle table layout (cplx entries): pass 1 [k-1][p] (k = 1..R1-1, p < S1), then pass 2 [k-1][p] (p < S2)
    static constexpr int TW1 = (R1 - 1) * S1;
    static constexpr int TW2 = (R2 > 1) ? (R2 - 1) * S2 : 0;
    static constexpr int TW_TOTAL = TW1 + TW2;
    // padded length of one line in shared memory (x pass): one pad every R3 and every R2*R3 elements
    static constexpr int PAD2 = (R2 > 1) ? S1 : (1 << 30);
    static constexpr int NPAD = N + N / R3 + ((R2 > 1) ? N / S1 : 0) + 1;
    static CANS_HD int pad(int e) { return e + e / R3 + ((R2 > 1) ? e / S1 : 0); }
    static CANS_HD int loc_of_freq(int q) {          // digit reversal
        int b = q % R1;
        int r = q / R1;
        int b2 = r % R2;
        int b3 = r / R2;
        return b * S1 + b2 * R3 + b3;
    }
};

// One butterfly task of a pass.  M = current sub-transform length, R = radix, S = M/R.
// `at(e)` maps a line location to the shared-memory element; `twp` points at this pass's [k-1][p] table.
template <int M, int R, bool INV, class At>
CANS_HD void fft_task(cplx* sm, const cplx* twp, int g, At at) {
    constexpr int S = M / R;
    const int blk = g / S;
    const int p = g - blk * S;
    const int base = blk * M + p;
    cplx v[R];
#pragma unroll
    for (int a = 0; a < R; ++a) v[a] = sm[at(base + S * a)];
    if (!INV) {
        Dft<R, false>::run(v);
        if (S > 1) {
#pragma unroll
            for (int k = 1; k < R; ++k) v[k] = cmul(v[k], twp[(k - 1) * S + p]);
        }
    } else {
        if (S > 1) {
#pragma unroll
            for (int k = 1; k < R; ++k) v[k] = cmulc(v[k], twp[(k - 1) * S + p]);
        }
        Dft<R, true>::run(v);
    }
#pragma unroll
    for (int a = 0; a < R; ++a) sm[at(base + S * a)] = v[a];
}

}  // namespace cans
