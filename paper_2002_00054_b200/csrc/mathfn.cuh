// mathfn.cuh -- the CUDA path's own FP64 special functions for the symmetry-function kernels.
//
// Why not libdevice exp / sincospi / sqrt here: ncu (profiles/r1_*) shows the hot loops are
// issue-bound, not FP64-pipe bound, and ~25 % of the issued instructions were UMOV / IMAD.MOV
// pairs materialising libdevice's 64-bit polynomial constants as immediates plus the
// BSSY/BSYNC/FSEL scaffolding of its special-case paths.  Here the coefficients live in the
// constant bank (DFMA takes c[bank][offset] operands directly), arguments are known to be
// in range, and the cosine cutoff is evaluated as a function of c^2 -- no sqrt, no rsqrt, no
// sincospi per triplet:
//     z = (pi c / (2 rc))^2 ,  C = cos(sqrt z) ,  S = sin(sqrt z)/sqrt z     (entire in z)
//     fc(c)    = (cos(pi c / rc) + 1)/2 = C^2
//     fc'(c)/c = -2 (pi/(2 rc))^2 C S
// Coefficients: coeffs.inc, written by gen_coeffs.py (Chebyshev-node fits; exp 1.2e-17, cos 2.0e-15 and
// sinc 1.4e-16 absolute -- degree 7 for the cutoff pair: four orders below the 1e-11 tolerance on G).
#pragma once

namespace nnp {

#include "coeffs.inc"

// exp(y) for y in [-700, 0.35]  (callers guarantee the range; no overflow / denormal handling).
__device__ __forceinline__ double exp_small(double y) {
    const double MAGIC = 6755399441055744.0;                 // 1.5 * 2^52: round-to-nearest-integer trick
    const double t = fma(y, 1.4426950408889634, MAGIC);      // y * log2(e)
    const int k = __double2loint(t);
    const double kf = t - MAGIC;
    double r = fma(kf, -6.93147180369123816490e-01, y);      // ln2 hi
    r = fma(kf, -1.90821492927058770002e-10, r);             // ln2 lo
    double p = EXPC[11];
#pragma unroll
    for (int q = 10; q >= 0; --q) p = fma(p, r, EXPC[q]);
    return __hiloint2double(__double2hiint(p) + (k << 20), __double2loint(p));
}

// exp(y) for y in [-0.05, 0]: no range reduction, degree 6.  The triplet Gaussian exp(-eta_0 c^2) of a
// model with eta_0 rc^2 <= 0.05 (the water-like models: 0.001 * 36) never leaves this interval.
__device__ __forceinline__ double exp_tiny(double y) {
    double p = EXPT[6];
#pragma unroll
    for (int q = 5; q >= 0; --q) p = fma(p, y, EXPT[q]);
    return p;
}

// the same with degree 5 (max error 1.0e-14 on [-0.05, 0]): the per-triplet Gaussian exp(-eta_0 c^2) of both hot kernels --
// one DFMA less in the dependent chain of every triplet; the per-neighbour staging keeps degree 6
__device__ __forceinline__ double exp_tiny5(double y) {
    double p = EXPT5[5];
#pragma unroll
    for (int q = 4; q >= 0; --q) p = fma(p, y, EXPT5[q]);
    return p;
}
__device__ __forceinline__ float exp_tiny5(float y) { return __expf(y); }

// C = cos(sqrt z), S = sin(sqrt z)/sqrt z for z in [0, (pi/2)^2]
__device__ __forceinline__ void cos_sinc(double z, double& C, double& S) {
    double c = COSC[7], s = SNCC[7];
#pragma unroll
    for (int q = 6; q >= 0; --q) {
        c = fma(c, z, COSC[q]);
        s = fma(s, z, SNCC[q]);
    }
    C = c;
    S = s;
}

__device__ __forceinline__ double cos_only(double z) {
    double c = COSC[7];
#pragma unroll
    for (int q = 6; q >= 0; --q) c = fma(c, z, COSC[q]);
    return c;
}

// ---- FP32 versions for the opt-in mixed-precision mode (nnp_set_precision): degree-5 cutoff
// polynomials (COSF / SNCF, 3e-8 absolute) and the hardware exponential ex2.approx (2 ulp); errors far below the FP32
// rounding of the sums they feed.
__device__ __forceinline__ float exp_small(float y) { return __expf(y); }
__device__ __forceinline__ float exp_tiny(float y) { return __expf(y); }
__device__ __forceinline__ void cos_sinc(float z, float& C, float& S) {
    float c = COSF[5], s = SNCF[5];
#pragma unroll
    for (int q = 4; q >= 0; --q) {
        c = fmaf(c, z, COSF[q]);
        s = fmaf(s, z, SNCF[q]);
    }
    C = c;
    S = s;
}
__device__ __forceinline__ float cos_only(float z) {
    float c = COSF[5];
#pragma unroll
    for (int q = 4; q >= 0; --q) c = fmaf(c, z, COSF[q]);
    return c;
}

// Cutoff of an SF with its own radius rc_s (nnp_set_sf_cutoffs), from r^2: fc = cos^2(pi r / (2 rc_s)) for
// r < rc_s, else 0; rc2 = rc_s^2, k2 = (pi / (2 rc_s))^2.  The polynomial argument is clamped to its range.
__device__ __forceinline__ double fc_own(double r2, double rc2, double k2) {
    const double C = cos_only(fmin(r2, rc2) * k2);
    return r2 < rc2 ? C * C : 0.0;
}

// the same with df = fc'(r) / r
__device__ __forceinline__ void fc_dfc_own(double r2, double rc2, double k2, double& f, double& df) {
    double C, S;
    cos_sinc(fmin(r2, rc2) * k2, C, S);
    const bool in = r2 < rc2;
    f = in ? C * C : 0.0;
    df = in ? (-2.0 * k2) * (C * S) : 0.0;
}

// x^n, n >= 1 an integer that is the same in every lane: square-and-multiply in a warp-uniform loop
// (the base exponent zeta0 of a free-eta pass, nnp_internal.h AngPass)
template <class R>
__device__ __forceinline__ R powi_uniform(R x, int n) {
    R r = (n & 1) ? x : (R)1;
    for (n >>= 1; n; n >>= 1) {
        x *= x;
        if (n & 1) r *= x;
    }
    return r;
}

}  // namespace nnp
