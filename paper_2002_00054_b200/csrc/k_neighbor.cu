// k_neighbor.cu -- S1: full neighbour list N(i) = { j != i : |r_j - r_i|_min-image^2 < rc^2 }
// from the (element, cell)-sorted SoA positions ("neighbor list", L116 "random
// access (neighbor list)").  One warp per atom; the <= 18 contiguous x-runs of the 3x3(x3) cell
// stencil are walked as one flat candidate range, hits are ballot-compacted and the row written coalesced.  Rows hold
// positions in the SORTED order, grouped by neighbour element (all of element 0, then 1, ...),
// which is what lets the symmetry-function kernels run type-homogeneous segments.
#include "geometry.cuh"
#include "nnp_internal.h"

namespace nnp {

constexpr int NB_WARPS = 8;

// distinct periodic cells {c-1, c, c+1} along one dimension (all cells if nc <= 3)
__device__ __forceinline__ int stencil_1d(int c, int nc, int* out) {
    if (nc <= 3) {
        for (int k = 0; k < nc; ++k) out[k] = k;
        return nc;
    }
    out[0] = (c == 0) ? nc - 1 : c - 1;
    out[1] = c;
    out[2] = (c == nc - 1) ? 0 : c + 1;
    return 3;
}

__global__ void __launch_bounds__(NB_WARPS * 32)
k_neighbors(int64_t n, int n_elem, Grid g, double rc2, int stride, int max_nbr,
            const double* __restrict__ sx, const double* __restrict__ sy, const double* __restrict__ sz,
            const int32_t* __restrict__ cell_start, int32_t* __restrict__ nbr, int32_t* __restrict__ nbr_cnt,
            int32_t* __restrict__ status, int32_t* __restrict__ sticky) {
    const int lane = threadIdx.x & 31;
    const int64_t i = (int64_t)blockIdx.x * NB_WARPS + (threadIdx.x >> 5);
    if (i >= n) return;
    const double xi = sx[i], yi = sy[i], zi = sz[i];
    int cx = (int)(xi * g.inv_cs[0]), cy = (int)(yi * g.inv_cs[1]), cz = (int)(zi * g.inv_cs[2]);
    cx = min(max(cx, 0), g.nc[0] - 1);
    cy = min(max(cy, 0), g.nc[1] - 1);
    cz = min(max(cz, 0), g.nc[2] - 1);
    int ys[3], zs[3];
    const int ny = stencil_1d(cy, g.nc[1], ys);
    const int nz = stencil_1d(cz, g.nc[2], zs);
    // x-runs: cells contiguous in memory -> at most two [first, last] cell ranges
    int xr0[2], xr1[2], nxr;
    if (g.nc[0] <= 3) { xr0[0] = 0; xr1[0] = g.nc[0] - 1; nxr = 1; }
    else if (cx == 0) { xr0[0] = 0; xr1[0] = 1; xr0[1] = g.nc[0] - 1; xr1[1] = g.nc[0] - 1; nxr = 2; }
    else if (cx == g.nc[0] - 1) { xr0[0] = 0; xr1[0] = 0; xr0[1] = cx - 1; xr1[1] = cx; nxr = 2; }
    else { xr0[0] = cx - 1; xr1[0] = cx + 1; nxr = 1; }

    // An atom of an interior cell (and >= 4 cells along the dimension) never needs the +-L of the minimum
    // image: its candidates are less than two cell widths <= L/2 away, so both conditions of min_image_1d
    // are false and the raw difference IS the result (same bits).  Warp-uniform -> 12 instructions fewer
    // per chunk of candidates for ~87 % of the atoms (the kernel is issue-bound: ncu, 83 % issue slots).
    const bool wx = !(g.nc[0] >= 4 && cx >= 1 && cx <= g.nc[0] - 2);
    const bool wy = !(g.nc[1] >= 4 && cy >= 1 && cy <= g.nc[1] - 2);
    const bool wz = !(g.nc[2] >= 4 && cz >= 1 && cz <= g.nc[2] - 2);
    int32_t* row = nbr + (size_t)i * stride;
    int cnt = 0;
    const int nrun = nz * ny * nxr;                     // <= 18 contiguous runs of candidates per element
    for (int e = 0; e < n_elem; ++e) {
        const int32_t* cs = cell_start + (size_t)e * g.ncell;
        const int cnt_before = cnt;
        // run table: lane r owns run r (its bounds come in ONE round trip instead of one per run), then the
        // candidates of all runs are walked as one flat index space -> full chunks of 32 whatever the run lengths
        int j0 = 0, len = 0;
        if (lane < nrun) {
            const int r = lane % nxr, ab = lane / nxr;
            const int b = ab % ny, a = ab / ny;
            const int rowbase = (zs[a] * g.nc[1] + ys[b]) * g.nc[0];
            j0 = cs[rowbase + xr0[r]];
            len = cs[rowbase + xr1[r] + 1] - j0;
        }
        int incl = len;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += t;
        }
        const int P = incl - len;                       // first flat index of run `lane`
        const int total = __shfl_sync(0xffffffffu, incl, 31);
        for (int f0 = 0; f0 < total; f0 += 32) {
            const int f = f0 + lane;
            int lo = 0, hi = 31;                        // largest run r with P[r] <= f
#pragma unroll
            for (int step = 0; step < 5; ++step) {
                const int mid = (lo + hi + 1) >> 1;
                const int pm = __shfl_sync(0xffffffffu, P, mid);
                if (pm <= f) lo = mid; else hi = mid - 1;
            }
            const int j = __shfl_sync(0xffffffffu, j0, lo) + (f - __shfl_sync(0xffffffffu, P, lo));
            bool hit = false;
            if (f < total && j != i) {
                const double dx = wx ? min_image_1d(xi, sx[j], g.box[0], g.half[0]) : __dsub_rn(sx[j], xi);
                const double dy = wy ? min_image_1d(yi, sy[j], g.box[1], g.half[1]) : __dsub_rn(sy[j], yi);
                const double dz = wz ? min_image_1d(zi, sz[j], g.box[2], g.half[2]) : __dsub_rn(sz[j], zi);
                hit = dist2_exact(dx, dy, dz) < rc2;
            }
            const unsigned m = __ballot_sync(0xffffffffu, hit);
            if (hit) {
                const int p = cnt + __popc(m & ((1u << lane) - 1u));
                if (p < max_nbr) row[p] = j;
            }
            cnt += __popc(m);
        }
        if (lane == 0) nbr_cnt[(size_t)i * MAX_ELEM + e] = min(cnt, max_nbr) - min(cnt_before, max_nbr);
    }
    if (lane == 0) {
        for (int e = n_elem; e < MAX_ELEM; ++e) nbr_cnt[(size_t)i * MAX_ELEM + e] = 0;
        if (cnt > max_nbr) { atomicOr(status, ST_NBR_OVERFLOW); atomicOr(sticky, ST_NBR_OVERFLOW); }
    }
}

int launch_neighbors(const Workspace& w, const Grid& g, int64_t n, int n_elem, double rc2, int stride,
                     int max_nbr, cudaStream_t st) {
    if (n == 0) return 0;
    const unsigned nb = (unsigned)((n + NB_WARPS - 1) / NB_WARPS);
    k_neighbors<<<nb, NB_WARPS * 32, 0, st>>>(n, n_elem, g, rc2, stride, max_nbr, w.sx, w.sy, w.sz, w.cell_start,
                                              w.nbr, w.nbr_cnt, w.status, w.sticky);
    return 1;
}

}  // namespace nnp
