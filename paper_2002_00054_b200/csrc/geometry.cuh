// geometry.cuh -- periodic-box arithmetic of the CUDA path (readings 1, C6, C7).
// The neighbour predicate must give the SAME bits as the definition, so every product and
// sum is an explicitly rounded intrinsic (nvcc would otherwise contract a*b+c into an FMA):
//   wrap:       w  = x - L*floor(x/L)
//   min image:  d  = w_j - w_i ; if (d > L/2) d -= L ; else if (d < -L/2) d += L
//   distance:   r2 = (dx*dx + dy*dy) + dz*dz ,   neighbour  <=>  r2 < rc*rc  (strict)
#pragma once
#include "nnp_internal.h"

namespace nnp {

__device__ __forceinline__ double wrap_coord(double x, double L) {
    const double q = floor(__ddiv_rn(x, L));
    return __dsub_rn(x, __dmul_rn(L, q));
}

__device__ __forceinline__ double min_image_1d(double xi, double xj, double L, double half) {
    double t = __dsub_rn(xj, xi);
    if (t > half) t = __dsub_rn(t, L);
    else if (t < -half) t = __dadd_rn(t, L);
    return t;
}

__device__ __forceinline__ double dist2_exact(double dx, double dy, double dz) {
    return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
}

// cell of a wrapped coordinate triple; the wrapped value may equal L (x = -tiny), hence the clamp
__device__ __forceinline__ int cell_of(double wx, double wy, double wz, const Grid& g) {
    int cx = (int)(wx * g.inv_cs[0]), cy = (int)(wy * g.inv_cs[1]), cz = (int)(wz * g.inv_cs[2]);
    cx = min(max(cx, 0), g.nc[0] - 1);
    cy = min(max(cy, 0), g.nc[1] - 1);
    cz = min(max(cz, 0), g.nc[2] - 1);
    return (cz * g.nc[1] + cy) * g.nc[0] + cx;
}

}  // namespace nnp
