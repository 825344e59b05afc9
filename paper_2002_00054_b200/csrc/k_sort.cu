// k_sort.cu -- S0 of the hot path: wrap positions into the box, bin them into cells and
// counting-sort the atoms by (element, cell, original index) into SoA arrays, so that
// every later kernel reads neighbour coordinates from a few contiguous runs (coalesced,
// L2-resident).  Also the prefix scans used here and by the exports.
//
// Geometry arithmetic follows DESIGN.md reading C7 exactly (every product and sum rounded
// on its own, no FMA contraction) because neighbour SETS must match the oracle bit for bit.
#include "geometry.cuh"
#include "nnp_internal.h"

namespace nnp {

// ---------------------------------------------------------------- exclusive scans

constexpr int SCAN_THREADS = 1024;
constexpr int SCAN_ITEMS = 4;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

// Block-level exclusive scan of up to SCAN_TILE elements per block; block total -> sums[block].
// `cond` (here and in the sort kernels below): null, or a device word -- the kernel returns at once when it is 0.
// The neighbour-skin mode (nnp_set_neighbor_skin) decides ON THE DEVICE whether a call rebuilds the sorted order and the
// candidate list, so the launch sequence of a call is always the same (CUDA-graph replay of nnp_md_run).
template <typename T>
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_tile(T* data, int64_t n, T* sums, const int32_t* __restrict__ cond) {
    __shared__ T warp_tot[32];
    if (cond && *cond == 0) return;
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    T v[SCAN_ITEMS];
    T tsum = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        v[k] = (base + k < n) ? data[base + k] : T(0);
        tsum += v[k];
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    T inc = tsum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        T t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
    }
    if (lane == 31) warp_tot[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        T w = warp_tot[lane];
        T winc = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            T t = __shfl_up_sync(0xffffffffu, winc, d);
            if (lane >= d) winc += t;
        }
        warp_tot[lane] = winc - w;   // exclusive warp offsets
        if (lane == 31 && sums) sums[blockIdx.x] = winc;
    }
    __syncthreads();
    T run = warp_tot[wid] + (inc - tsum);
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        if (base + k < n) data[base + k] = run;
        run += v[k];
    }
}

template <typename T>
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_add(T* data, int64_t n, const T* sums, const int32_t* __restrict__ cond) {
    if (cond && *cond == 0) return;
    const T off = sums[blockIdx.x];
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k)
        if (base + k < n) data[base + k] += off;
}

// In-place exclusive scan of data[0..n); tmp needs >= n/SCAN_TILE + 2*SCAN_TILE + 2 entries.
template <typename T>
static void scan_rec(T* data, int64_t n, T* tmp, cudaStream_t st, int* launches, const int32_t* cond = nullptr) {
    if (n <= 0) return;
    const int64_t nb = (n + SCAN_TILE - 1) / SCAN_TILE;
    if (nb == 1) {
        k_scan_tile<T><<<1, SCAN_THREADS, 0, st>>>(data, n, nullptr, cond);
        ++*launches;
        return;
    }
    k_scan_tile<T><<<(unsigned)nb, SCAN_THREADS, 0, st>>>(data, n, tmp, cond);
    ++*launches;
    scan_rec<T>(tmp, nb, tmp + nb, st, launches, cond);
    k_scan_add<T><<<(unsigned)nb, SCAN_THREADS, 0, st>>>(data, n, tmp, cond);
    ++*launches;
}

void exclusive_scan_i32(int32_t* d_data, int64_t n, int32_t* d_tmp, cudaStream_t st, int* launches) {
    scan_rec<int32_t>(d_data, n, d_tmp, st, launches);
}

__global__ void k_widen(const int32_t* in, int64_t n, int64_t* out) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = in[i];
    if (i == n) out[n] = 0;
}

int launch_scan_i64_from_i32(const int32_t* d_in, int64_t n, int64_t* d_out, int64_t* d_tmp, cudaStream_t st) {
    int launches = 0;
    k_widen<<<(unsigned)((n + 1 + 255) / 256), 256, 0, st>>>(d_in, n, d_out);
    ++launches;
    scan_rec<int64_t>(d_out, n + 1, d_tmp, st, &launches);
    return launches;
}

// ---------------------------------------------------------------- binning + sort

// key = element * ncell + cell; rank = arrival order inside the key (made deterministic later).
__global__ void k_zero_i32(int32_t* __restrict__ data, int64_t n, const int32_t* __restrict__ cond) {
    if (cond && *cond == 0) return;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) data[i] = 0;
}

__global__ void k_bin(int64_t n, const double* __restrict__ pos, const int32_t* __restrict__ type, Grid g,
                      int n_elem, int32_t* __restrict__ key, int32_t* __restrict__ rank,
                      int32_t* __restrict__ cell_cnt, int32_t* __restrict__ status, int32_t* __restrict__ sticky,
                      const int32_t* __restrict__ cond) {
    if (cond && *cond == 0) return;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
    int t = type[i];
    int bad = 0;
    if (!(isfinite(x) && isfinite(y) && isfinite(z))) bad |= ST_NONFINITE;
    if (t < 0 || t >= n_elem) { bad |= ST_TYPE_RANGE; t = 0; }
    if (bad) { atomicOr(status, bad); atomicOr(sticky, bad); }
    const double wx = (bad & ST_NONFINITE) ? 0.0 : wrap_coord(x, g.box[0]);
    const double wy = (bad & ST_NONFINITE) ? 0.0 : wrap_coord(y, g.box[1]);
    const double wz = (bad & ST_NONFINITE) ? 0.0 : wrap_coord(z, g.box[2]);
    const int c = cell_of(wx, wy, wz, g);
    const int k = t * g.ncell + c;
    key[i] = k;
    rank[i] = atomicAdd(&cell_cnt[k], 1);
}

__global__ void k_scatter(int64_t n, const double* __restrict__ pos, Grid g, const int32_t* __restrict__ key,
                          const int32_t* __restrict__ rank, const int32_t* __restrict__ cell_start,
                          double* __restrict__ tx, double* __restrict__ ty, double* __restrict__ tz,
                          int32_t* __restrict__ tperm, int32_t* __restrict__ tkey, const int32_t* __restrict__ cond) {
    if (cond && *cond == 0) return;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int k = key[i];
    const int dst = cell_start[k] + rank[i];
    const double x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
    const bool ok = isfinite(x) && isfinite(y) && isfinite(z);
    tx[dst] = ok ? wrap_coord(x, g.box[0]) : 0.0;
    ty[dst] = ok ? wrap_coord(y, g.box[1]) : 0.0;
    tz[dst] = ok ? wrap_coord(z, g.box[2]) : 0.0;
    tperm[dst] = (int32_t)i;
    tkey[dst] = k;
}

// Order the atoms of every (element, cell) bucket by original index, so the sorted order -- and
// with it every neighbour-row order and floating-point summation order downstream -- does not
// depend on the arrival order of the atomics in k_bin.
__global__ void k_cell_order(int64_t n, const int32_t* __restrict__ cell_start, const int32_t* __restrict__ tkey,
                             const int32_t* __restrict__ tperm, const double* __restrict__ tx,
                             const double* __restrict__ ty, const double* __restrict__ tz,
                             double* __restrict__ sx, double* __restrict__ sy, double* __restrict__ sz,
                             int32_t* __restrict__ perm, double* __restrict__ bx, double* __restrict__ by,
                             double* __restrict__ bz, const int32_t* __restrict__ cond) {
    if (cond && *cond == 0) return;
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const int k = tkey[p];
    const int s = cell_start[k], e = cell_start[k + 1];
    const int me = tperm[p];
    int r = 0;
    for (int q = s; q < e; ++q) r += (tperm[q] < me);
    const int dst = s + r;
    sx[dst] = tx[p];
    sy[dst] = ty[p];
    sz[dst] = tz[p];
    perm[dst] = me;
    if (bx) {                    // neighbour-skin mode: the positions the candidate list is built from
        bx[dst] = tx[p];
        by[dst] = ty[p];
        bz[dst] = tz[p];
    }
}

// ---------------------------------------------------------------- neighbour-skin mode: reuse of the sorted order
// (SURVEY.md 8(f)1 / PAPER.md L48: the neighbour list of an MD code is rebuilt only every few steps.)
// k_skin_check: does the candidate list of the last rebuild (radius rc + skin) still hold every pair within rc?  Yes as
// long as no atom has moved more than skin/2 from its position at the rebuild (two atoms approach by at most skin) and
// every atom still has the element it was sorted under.  Sets *flag to 1 otherwise; a non-finite position also lands
// here (the comparison is written so that a NaN fails it) and is then reported by k_bin.
__global__ void k_skin_check(int64_t n, const double* __restrict__ pos, const int32_t* __restrict__ type,
                             const int32_t* __restrict__ perm, const double* __restrict__ bx,
                             const double* __restrict__ by, const double* __restrict__ bz, Grid g, int n_elem,
                             const int32_t* __restrict__ cell_start, double lim2, int32_t* __restrict__ flag) {
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const int32_t i = perm[p];
    bool bad = i < 0 || i >= n;
    if (!bad) {
        int t = 0;
        for (int e = 1; e < n_elem; ++e)
            if (p >= cell_start[(size_t)e * g.ncell]) t = e;
        bad = type[i] != t;
        const double dx = min_image_1d(bx[p], wrap_coord(pos[3 * (size_t)i], g.box[0]), g.box[0], g.half[0]);
        const double dy = min_image_1d(by[p], wrap_coord(pos[3 * (size_t)i + 1], g.box[1]), g.box[1], g.half[1]);
        const double dz = min_image_1d(bz[p], wrap_coord(pos[3 * (size_t)i + 2], g.box[2]), g.box[2], g.half[2]);
        bad |= !(dist2_exact(dx, dy, dz) <= lim2);
    }
    if (bad) *flag = 1;
}

// a call that keeps the sorted order: the current (wrapped) positions in that order
__global__ void k_regather(int64_t n, const double* __restrict__ pos, const int32_t* __restrict__ perm, Grid g,
                           double* __restrict__ sx, double* __restrict__ sy, double* __restrict__ sz,
                           const int32_t* __restrict__ rebuild) {
    if (*rebuild != 0) return;
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const size_t i = (size_t)perm[p];
    sx[p] = wrap_coord(pos[3 * i], g.box[0]);
    sy[p] = wrap_coord(pos[3 * i + 1], g.box[1]);
    sz[p] = wrap_coord(pos[3 * i + 2], g.box[2]);
}

// skin_mode 0: plain sort (every call).  1: neighbour-skin mode, rebuild forced by the host (first call on this
// workspace, another n / box / setting).  2: neighbour-skin mode, the device decides (k_skin_check -> w.skin_flag);
// a call that keeps the order only re-gathers the positions.
int launch_sort(const Workspace& w, const Grid& g, int64_t n, int n_elem, const double* d_pos,
                const int32_t* d_type, int skin_mode, double skin, cudaStream_t st) {
    int launches = 0;
    const int64_t n_keys = (int64_t)n_elem * g.ncell;
    const unsigned nb = (unsigned)((n + 255) / 256);
    cudaMemsetAsync(w.status, 0, sizeof(int32_t) * 4, st);
    const int32_t* cond = nullptr;
    if (skin_mode == 0) {
        cudaMemsetAsync(w.cell_start, 0, sizeof(int32_t) * (size_t)(n_keys + 1), st);
    } else {
        cond = w.skin_flag;
        cudaMemsetAsync(w.skin_flag, skin_mode == 1 ? 1 : 0, sizeof(int32_t), st);     // any non-zero word means "rebuild"
        if (skin_mode == 2) {
            k_skin_check<<<nb, 256, 0, st>>>(n, d_pos, d_type, w.perm, w.bx, w.by, w.bz, g, n_elem, w.cell_start,
                                             0.25 * skin * skin, w.skin_flag);
            ++launches;
        }
        k_zero_i32<<<(unsigned)((n_keys + 1 + 255) / 256), 256, 0, st>>>(w.cell_start, n_keys + 1, cond);
        ++launches;
    }
    k_bin<<<nb, 256, 0, st>>>(n, d_pos, d_type, g, n_elem, w.key, w.rank, w.cell_start, w.status, w.sticky, cond);
    ++launches;
    scan_rec<int32_t>(w.cell_start, n_keys + 1, w.scan_tmp, st, &launches, cond);
    k_scatter<<<nb, 256, 0, st>>>(n, d_pos, g, w.key, w.rank, w.cell_start, w.tx, w.ty, w.tz, w.tperm, w.tkey, cond);
    ++launches;
    k_cell_order<<<nb, 256, 0, st>>>(n, w.cell_start, w.tkey, w.tperm, w.tx, w.ty, w.tz, w.sx, w.sy, w.sz, w.perm,
                                     skin_mode ? w.bx : nullptr, w.by, w.bz, cond);
    ++launches;
    if (skin_mode == 2) {
        k_regather<<<nb, 256, 0, st>>>(n, d_pos, w.perm, g, w.sx, w.sy, w.sz, w.skin_flag);
        ++launches;
    }
    return launches;
}

}  // namespace nnp
