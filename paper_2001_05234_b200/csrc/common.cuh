// common.cuh -- small helpers shared by the sm_100a kernels of libcans_poisson.
// Device code only (the CPU oracle shares nothing with this tree).
#pragma once

#if defined(__CUDACC__)
#include <cuda_runtime.h>
#define CANS_HD __host__ __device__ __forceinline__
#define CANS_D __device__ __forceinline__
#else
// Host-side syntax shim: lets a development harness type-check / single-step the index logic of
// the phase functions with a plain C++ compiler.  Never part of the shipped library.
#include <cmath>
struct double2 { double x, y; };
static inline double2 make_double2(double x, double y) { double2 r; r.x = x; r.y = y; return r; }
#define CANS_HD inline
#define CANS_D inline
#endif

namespace cans {

typedef double2 cplx;   // (re, im)

CANS_HD cplx cmk(double re, double im) { return make_double2(re, im); }
CANS_HD cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
CANS_HD cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
CANS_HD cplx cneg(cplx a) { return make_double2(-a.x, -a.y); }
CANS_HD cplx cconj(cplx a) { return make_double2(a.x, -a.y); }
CANS_HD cplx cscale(cplx a, double s) { return make_double2(a.x * s, a.y * s); }
// a * b
CANS_HD cplx cmul(cplx a, cplx b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
// a * conj(b)
CANS_HD cplx cmulc(cplx a, cplx b) {
    return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
// a * (-i)  and  a * (+i)
CANS_HD cplx cmul_mi(cplx a) { return make_double2(a.y, -a.x); }
CANS_HD cplx cmul_pi(cplx a) { return make_double2(-a.y, a.x); }

// 16-byte load of the field being transformed in place.  L2-only (ld.global.cg): inside the fused
// persistent kernels the same addresses are rewritten by other CTAs between two reads of one SM, and
// L1 is not coherent; the data is streamed once per task, so L1 would not help anyway.
CANS_HD double2 ld_p2(const double* p) {
#if defined(__CUDA_ARCH__)
    return __ldcg(reinterpret_cast<const double2*>(p));
#else
    return *reinterpret_cast<const double2*>(p);
#endif
}

// 16-byte load of data that is streamed once (u, v, w of the fused divergence).  A plain load: the L2-only variants
// (ld.global.cg / .cs) were measured on the C5 grid and changed nothing, the twiddle tables stay in L1 either way.
CANS_HD double2 ldg_stream2(const double* p) { return *reinterpret_cast<const double2*>(p); }

// Transform kind of one direction (pressure boundary pair), see DESIGN.md "Transforms".
// KIND_ND / KIND_DN: the mixed pairs (lower Neumann, upper Dirichlet and the reverse), DCT-IV / DST-IV.
enum Kind : int { KIND_PP = 0, KIND_NN = 1, KIND_DD = 2, KIND_ND = 3, KIND_DN = 4 };
CANS_HD bool kind_mixed(int kind) { return kind >= KIND_ND; }
// odd samples enter the FFT negated
CANS_HD bool kind_neg_odd(int kind) { return kind == KIND_DD || kind == KIND_ND; }

}  // namespace cans
