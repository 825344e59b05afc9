// k_neighbor.cu -- S1: full neighbour list N(i) = { j != i : |r_j - r_i|_min-image^2 < rc^2 }
// from the (element, cell)-sorted SoA positions ("neighbor list", L116 "random
// access (neighbor list)").  One warp per cell; cells are rc / HW wide (HW = Grid::hw: 2, or 1 for sparse cells) and the <= (2 HW + 1)^2 contiguous x-runs of the
// cell stencil are walked as one flat candidate range, hits are ballot-compacted and the row written coalesced.  Rows hold
// positions in the SORTED order, grouped by neighbour element (all of element 0, then 1, ...),
// which is what lets the symmetry-function kernels run type-homogeneous segments.
#include "geometry.cuh"
#include "nnp_internal.h"

namespace nnp {

constexpr int NB_WARPS = 8;

// distinct periodic cells {c-HW .. c+HW} along one dimension (all cells if nc <= 2 HW + 1)
template <int HW>                               // cells are >= rc / HW wide (make_grid)
__device__ __forceinline__ int stencil_1d(int c, int nc, int* out) {
    constexpr int SW = 2 * HW + 1;
    if (nc <= SW) {
        for (int k = 0; k < nc; ++k) out[k] = k;
        return nc;
    }
#pragma unroll
    for (int k = 0; k < SW; ++k) {
        int q = c + k - HW;
        if (q < 0) q += nc;
        if (q >= nc) q -= nc;
        out[k] = q;
    }
    return SW;
}

// One warp per CELL: the atoms of a cell (all elements) share their stencil, so the run table, the flat candidate
// index and the candidate loads are done once per chunk of 32 candidates and every centre of the cell tests the chunk
// from registers (one atom per warp spent ~2/3 of its instructions on exactly that bookkeeping: 4.5 ms at 2.1 M atoms).
// The centres' coordinates, row offsets and running counts sit in shared memory and are read as broadcasts.  A cell whose stencil
// does not wrap (87 % of the cells of a 2.1 M-atom box) takes a branch-free test on raw differences (4.5 -> 3.33 -> 2.63 ms).
template <int HW>
__global__ void __launch_bounds__(NB_WARPS * 32)
k_neighbors(int64_t n, int n_elem, Grid g, double rc2, int stride, int max_nbr,
            const double* __restrict__ sx, const double* __restrict__ sy, const double* __restrict__ sz,
            const int32_t* __restrict__ cell_start, int32_t* __restrict__ nbr, int32_t* __restrict__ nbr_cnt,
            int32_t* __restrict__ status, int32_t* __restrict__ sticky, const int32_t* __restrict__ cond) {
    if (cond && *cond == 0) return;          // neighbour-skin mode: the candidate list of an earlier call still holds
    constexpr int SW = 2 * HW + 1;
    __shared__ double cpos[NB_WARPS][3][32];
    __shared__ int32_t cidx[NB_WARPS][32];
    __shared__ int32_t ccnt[NB_WARPS][32];       // neighbours found so far, per centre of the group
    __shared__ size_t crow[NB_WARPS][32];        // first entry of the centre's row
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t c = (int64_t)blockIdx.x * NB_WARPS + wid;
    if (c >= g.ncell) return;
    const int cx = (int)(c % g.nc[0]), cy = (int)((c / g.nc[0]) % g.nc[1]), cz = (int)(c / ((int64_t)g.nc[0] * g.nc[1]));
    // the centres of this cell: element-major ranges of the sorted order
    int cb[MAX_ELEM + 1];
    int first[MAX_ELEM];
    cb[0] = 0;
#pragma unroll
    for (int e = 0; e < MAX_ELEM; ++e) {
        int lo = 0, hi = 0;
        if (e < n_elem) { lo = cell_start[(size_t)e * g.ncell + c]; hi = cell_start[(size_t)e * g.ncell + c + 1]; }
        first[e] = lo;
        cb[e + 1] = cb[e] + (hi - lo);
    }
    const int n_centres = cb[MAX_ELEM];
    if (n_centres == 0) return;
    int ys[SW], zs[SW];
    const int ny = stencil_1d<HW>(cy, g.nc[1], ys);
    const int nz = stencil_1d<HW>(cz, g.nc[2], zs);
    // x-runs: cells contiguous in memory -> at most two [first, last] cell ranges
    int xr0[2], xr1[2], nxr = 1;
    if (g.nc[0] <= SW) { xr0[0] = 0; xr1[0] = g.nc[0] - 1; }
    else if (cx < HW) { xr0[0] = 0; xr1[0] = cx + HW; xr0[1] = g.nc[0] + cx - HW; xr1[1] = g.nc[0] - 1; nxr = 2; }
    else if (cx + HW >= g.nc[0]) { xr0[0] = 0; xr1[0] = cx + HW - g.nc[0]; xr0[1] = cx - HW; xr1[1] = g.nc[0] - 1; nxr = 2; }
    else { xr0[0] = cx - HW; xr1[0] = cx + HW; }
    // A cell whose stencil does not wrap (and >= 2 SW cells along the dimension) never needs the +-L of the minimum
    // image: the candidates are less than HW + 1 cell widths <= L/2 away, so both conditions of min_image_1d are
    // false and the raw difference IS the result (same bits).
    const bool wx = !(g.nc[0] >= 2 * SW && cx >= HW && cx + HW < g.nc[0]);
    const bool wy = !(g.nc[1] >= 2 * SW && cy >= HW && cy + HW < g.nc[1]);
    const bool wz = !(g.nc[2] >= 2 * SW && cz >= HW && cz + HW < g.nc[2]);
    const int nyz = nz * ny;                            // <= SW^2 <= 25 contiguous runs of candidates per element and x-range

    for (int g0 = 0; g0 < n_centres; g0 += 32) {        // groups of 32 centres (one group unless the cell is very dense)
        const int ng = min(32, n_centres - g0);
        int my = -1;                                    // sorted index of the centre this lane keeps the counters of
        if (lane < ng) {
            const int q = g0 + lane;
            int e = 0;
#pragma unroll
            for (int k = 1; k < MAX_ELEM; ++k)
                if (q >= cb[k]) e = k;
            my = first[e] + (q - cb[e]);
            cpos[wid][0][lane] = sx[my]; cpos[wid][1][lane] = sy[my]; cpos[wid][2][lane] = sz[my];
        }
        cidx[wid][lane] = my;
        ccnt[wid][lane] = 0;
        crow[wid][lane] = (size_t)(my >= 0 ? my : 0) * stride;
        __syncwarp();
        int cnt = 0;                                    // lane a: neighbours of centre a found so far (copied from ccnt per element)
        for (int e = 0; e < n_elem; ++e) {
            const int32_t* cs = cell_start + (size_t)e * g.ncell;
            const int cnt_before = cnt;
            for (int r = 0; r < nxr; ++r) {
                // run table: lane q owns run q (its bounds come in ONE round trip instead of one per run), then the
                // candidates of all runs are walked as one flat index space -> full chunks of 32 whatever the run lengths
                int j0 = 0, len = 0;
                if (lane < nyz) {
                    const int b = lane % ny, a = lane / ny;
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
                    int lo = 0, hi = 31;                        // largest run q with P[q] <= f
#pragma unroll
                    for (int step = 0; step < 5; ++step) {
                        const int mid = (lo + hi + 1) >> 1;
                        const int pm = __shfl_sync(0xffffffffu, P, mid);
                        if (pm <= f) lo = mid; else hi = mid - 1;
                    }
                    const int j = __shfl_sync(0xffffffffu, j0, lo) + (f - __shfl_sync(0xffffffffu, P, lo));
                    const bool have = f < total;
                    double xj = 0.0, yj = 0.0, zj = 0.0;
                    if (have) { xj = sx[j]; yj = sy[j]; zj = sz[j]; }
                    const unsigned lt = (1u << lane) - 1u;
                    if (!(wx || wy || wz)) {
                        // a cell whose stencil does not wrap: raw differences, no branch in the test (a lane without a
                        // candidate holds (0, 0, 0): whatever it computes is masked by `have`)
                        for (int a = 0; a < ng; ++a) {
                            const int i = cidx[wid][a];
                            const double dx = __dsub_rn(xj, cpos[wid][0][a]), dy = __dsub_rn(yj, cpos[wid][1][a]),
                                         dz = __dsub_rn(zj, cpos[wid][2][a]);
                            const bool hit = have & (j != i) & (dist2_exact(dx, dy, dz) < rc2);
                            const unsigned m = __ballot_sync(0xffffffffu, hit);
                            const int base = ccnt[wid][a];
                            const int p = base + __popc(m & lt);
                            if (hit && p < max_nbr) nbr[crow[wid][a] + p] = j;
                            __syncwarp();
                            if (lane == 0) ccnt[wid][a] = base + __popc(m);
                        }
                        __syncwarp();
                    } else
                    for (int a = 0; a < ng; ++a) {              // every centre of the group against this chunk
                        const int i = cidx[wid][a];
                        const double xi = cpos[wid][0][a], yi = cpos[wid][1][a], zi = cpos[wid][2][a];
                        bool hit = false;
                        if (have && j != i) {
                            const double dx = wx ? min_image_1d(xi, xj, g.box[0], g.half[0]) : __dsub_rn(xj, xi);
                            const double dy = wy ? min_image_1d(yi, yj, g.box[1], g.half[1]) : __dsub_rn(yj, yi);
                            const double dz = wz ? min_image_1d(zi, zj, g.box[2], g.half[2]) : __dsub_rn(zj, zi);
                            hit = dist2_exact(dx, dy, dz) < rc2;
                        }
                        const unsigned m = __ballot_sync(0xffffffffu, hit);
                        const int base = ccnt[wid][a];
                        if (hit) {
                            const int p = base + __popc(m & ((1u << lane) - 1u));
                            if (p < max_nbr) nbr[(size_t)i * stride + p] = j;
                        }
                        __syncwarp();
                        if (lane == 0) ccnt[wid][a] = base + __popc(m);
                        __syncwarp();
                    }
                }
            }
            cnt = ccnt[wid][lane];
            if (my >= 0) nbr_cnt[(size_t)my * MAX_ELEM + e] = min(cnt, max_nbr) - min(cnt_before, max_nbr);
        }
        if (my >= 0) {
            for (int e = n_elem; e < MAX_ELEM; ++e) nbr_cnt[(size_t)my * MAX_ELEM + e] = 0;
            if (cnt > max_nbr) { atomicOr(status, ST_NBR_OVERFLOW); atomicOr(sticky, ST_NBR_OVERFLOW); }
        }
        __syncwarp();
    }
}

// Neighbour-skin mode, every call: the exact list N(i) of THIS call's positions, filtered from the candidate list
// (radius rc + skin, built by k_neighbors on the last rebuild) with the same FP64 predicate as a fresh build -- the
// symmetry-function and force kernels never see a slot beyond rc (staging the extra ~27 % of slots cost them 7x what
// a rebuild costs: DESIGN.md 11a).  A candidate row is grouped by element and so is the filtered row.  LPA lanes per
// atom, UN candidates per lane in flight (the loop is latency-bound; one chunk covers the short rows of a metal).
template <int LPA, int UN>
__global__ void __launch_bounds__(256)
k_filter(int64_t n, int n_elem, Grid g, double rc2, int sstride, int stride, int max_nbr,
         const double* __restrict__ sx, const double* __restrict__ sy, const double* __restrict__ sz,
         const int32_t* __restrict__ snbr, const int32_t* __restrict__ snbr_cnt, int32_t* __restrict__ nbr,
         int32_t* __restrict__ nbr_cnt, int32_t* __restrict__ status, int32_t* __restrict__ sticky,
         const int32_t* __restrict__ flag, int32_t* __restrict__ stats) {
    if (blockIdx.x == 0 && threadIdx.x == 0) {           // [0] calls, [1] rebuilds since nnp_set_neighbor_skin
        atomicAdd(&stats[0], 1);
        if (*flag != 0) atomicAdd(&stats[1], 1);
    }
    const int sub = threadIdx.x & (LPA - 1);
    const int64_t i = ((int64_t)blockIdx.x * 256 + threadIdx.x) / LPA;
    const unsigned gmask = LPA == 32 ? 0xffffffffu : (((1u << LPA) - 1u) << ((threadIdx.x & 31) & ~(LPA - 1)));
    const bool live = i < n;
    const int64_t ii = live ? i : n - 1;                 // idle groups of the last warp replay the last atom, writes off
    const double xi = sx[ii], yi = sy[ii], zi = sz[ii];
    const int32_t* __restrict__ srow = snbr + (size_t)ii * sstride;
    int32_t* __restrict__ row = nbr + (size_t)ii * stride;
    // the candidate row is packed: element e occupies [bnd[e], bnd[e+1])
    int bnd[MAX_ELEM + 1];
    bnd[0] = 0;
#pragma unroll
    for (int e = 0; e < MAX_ELEM; ++e) bnd[e + 1] = bnd[e] + (e < n_elem ? snbr_cnt[(size_t)ii * MAX_ELEM + e] : 0);
    const int tot = bnd[MAX_ELEM];
    int cnt = 0;
    int below[MAX_ELEM + 1];                             // hits among the candidates before bnd[e]
#pragma unroll
    for (int e = 0; e <= MAX_ELEM; ++e) below[e] = 0;
    // UN candidates per lane in flight: the loop is latency-bound
    for (int f0 = 0; f0 < tot; f0 += UN * LPA) {
        int j[UN];
        double x[UN], y[UN], z[UN];
#pragma unroll
        for (int u = 0; u < UN; ++u) {
            const int f = f0 + u * LPA + sub;
            j[u] = f < tot ? srow[f] : -1;
        }
#pragma unroll
        for (int u = 0; u < UN; ++u) {
            x[u] = y[u] = z[u] = 0.0;
            if (j[u] >= 0) { x[u] = sx[j[u]]; y[u] = sy[j[u]]; z[u] = sz[j[u]]; }
        }
#pragma unroll
        for (int u = 0; u < UN; ++u) {
            const int f = f0 + u * LPA + sub;
            const double dx = min_image_1d(xi, x[u], g.box[0], g.half[0]);
            const double dy = min_image_1d(yi, y[u], g.box[1], g.half[1]);
            const double dz = min_image_1d(zi, z[u], g.box[2], g.half[2]);
            const bool hit = j[u] >= 0 && dist2_exact(dx, dy, dz) < rc2;
            const unsigned m = __ballot_sync(gmask, hit);       // the groups of a warp run different trip counts
            if (hit && live) {
                const int p = cnt + __popc(m & ((1u << (threadIdx.x & 31)) - 1u));
                if (p < max_nbr) row[p] = j[u];
            }
            cnt += __popc(m);
#pragma unroll
            for (int e = 1; e <= MAX_ELEM; ++e) below[e] += __popc(__ballot_sync(gmask, hit && f < bnd[e]));
        }
    }
    if (sub == 0 && live) {
#pragma unroll
        for (int e = 0; e < MAX_ELEM; ++e)
            nbr_cnt[(size_t)i * MAX_ELEM + e] = min(below[e + 1], max_nbr) - min(below[e], max_nbr);
        if (cnt > max_nbr) { atomicOr(status, ST_NBR_OVERFLOW); atomicOr(sticky, ST_NBR_OVERFLOW); }
    }
}

// skin_mode 0: the exact list straight from the cells.  Otherwise: the candidate list (radius^2 rs2, rows of sstride,
// at most smax entries) if this call rebuilds, then the filter.
int launch_neighbors(const Workspace& w, const Grid& g, int64_t n, int n_elem, double rc2, int stride,
                     int max_nbr, int skin_mode, double rs2, int sstride, int smax, cudaStream_t st) {
    if (n == 0) return 0;
    const unsigned nb = (unsigned)((g.ncell + NB_WARPS - 1) / NB_WARPS);      // one warp per cell
    auto search = g.hw == 2 ? k_neighbors<2> : k_neighbors<1>;
    if (skin_mode == 0) {
        search<<<nb, NB_WARPS * 32, 0, st>>>(n, n_elem, g, rc2, stride, max_nbr, w.sx, w.sy, w.sz, w.cell_start,
                                             w.nbr, w.nbr_cnt, w.status, w.sticky, nullptr);
        return 1;
    }
    search<<<nb, NB_WARPS * 32, 0, st>>>(n, n_elem, g, rs2, sstride, smax, w.sx, w.sy, w.sz, w.cell_start,
                                         w.snbr, w.snbr_cnt, w.status, w.sticky, w.skin_flag);
#define NNP_FILTER(LPA, UN)                                                                                         \
    k_filter<LPA, UN><<<(unsigned)((n * LPA + 255) / 256), 256, 0, st>>>(n, n_elem, g, rc2, sstride, stride, max_nbr, w.sx, w.sy, \
                                                                         w.sz, w.snbr, w.snbr_cnt, w.nbr, w.nbr_cnt, w.status,   \
                                                                         w.sticky, w.skin_flag, w.skin_stats)
    if (smax <= 64) NNP_FILTER(32, 1);           // metals: ~26 candidates, one chunk
    else if (smax <= 128) NNP_FILTER(32, 2);
    else NNP_FILTER(32, 4);                      // water-like: ~120 candidates
#undef NNP_FILTER
    return 2;
}

}  // namespace nnp
