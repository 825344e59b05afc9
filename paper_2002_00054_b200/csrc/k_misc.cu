// k_misc.cu -- S5 (un-permute + deterministic energy reduction), the debug/parity exports and
// the FP64 issue-rate micro-benchmark used as roofline denominator.
#include "nnp_internal.h"

namespace nnp {

// ---------------------------------------------------------------- S5 finalize

constexpr int FIN_THREADS = 256;

// caller-order outputs + per-block partial sums of the atomic energies (sorted order, fixed tree)
__global__ void __launch_bounds__(FIN_THREADS)
k_unpermute(int64_t n, const int32_t* __restrict__ perm, const double* __restrict__ e_sorted,
            const double* __restrict__ f_sorted, double* __restrict__ e_atom, double* __restrict__ force,
            double* __restrict__ partial, int fixed) {
    __shared__ double red[FIN_THREADS];
    const int64_t p = (int64_t)blockIdx.x * FIN_THREADS + threadIdx.x;
    double e = 0.0;
    if (p < n) {
        const int64_t i = perm[p];
        e = e_sorted[p];
        e_atom[i] = e;
        if (fixed) {        // fixed-point sums of the deterministic mode (nnp_internal.h force_add)
            const unsigned long long* fb = reinterpret_cast<const unsigned long long*>(f_sorted);
            force[3 * i + 0] = force_from_fixed(fb[3 * p + 0]);
            force[3 * i + 1] = force_from_fixed(fb[3 * p + 1]);
            force[3 * i + 2] = force_from_fixed(fb[3 * p + 2]);
        } else {
            force[3 * i + 0] = f_sorted[3 * p + 0];
            force[3 * i + 1] = f_sorted[3 * p + 1];
            force[3 * i + 2] = f_sorted[3 * p + 2];
        }
    }
    red[threadIdx.x] = e;
    __syncthreads();
    for (int s = FIN_THREADS / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = red[0];
}

__global__ void __launch_bounds__(1024) k_sum_partials(int64_t nb, const double* __restrict__ partial,
                                                      double* __restrict__ e_total) {
    __shared__ double red[1024];
    double acc = 0.0;
    for (int64_t b = threadIdx.x; b < nb; b += 1024) acc += partial[b];   // fixed assignment -> deterministic
    red[threadIdx.x] = acc;
    __syncthreads();
    for (int s = 512; s > 0; s >>= 1) {
        if (threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) *e_total = red[0];
}

int launch_finalize(const Workspace& w, int64_t n, double* d_e_atom, double* d_e_total, double* d_force, int fixed_forces,
                    cudaStream_t st) {
    const int64_t nb = (n + FIN_THREADS - 1) / FIN_THREADS;
    int launches = 0;
    if (nb > 0) {
        k_unpermute<<<(unsigned)nb, FIN_THREADS, 0, st>>>(n, w.perm, w.e_sorted, w.f_sorted, d_e_atom, d_force, w.partial, fixed_forces);
        ++launches;
    }
    k_sum_partials<<<1, 1024, 0, st>>>(nb, w.partial, d_e_total);
    return launches + 1;
}

// ---------------------------------------------------------------- exports (caller's atom order)

__global__ void k_export_counts(int64_t n, int n_elem, const int32_t* __restrict__ perm,
                                const int32_t* __restrict__ nbr_cnt, int32_t* __restrict__ counts) {
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    int c = 0;
    for (int e = 0; e < n_elem; ++e) c += nbr_cnt[(size_t)p * MAX_ELEM + e];
    counts[perm[p]] = c;
}

int launch_export_counts(const Workspace& w, int64_t n, int n_elem, int32_t* d_counts, cudaStream_t st) {
    if (n == 0) return 0;
    k_export_counts<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, n_elem, w.perm, w.nbr_cnt, d_counts);
    return 1;
}

// one warp per row: map to original ids, bitonic-sort ascending in shared memory, write out
constexpr int EXP_WARPS = 4;
__global__ void __launch_bounds__(EXP_WARPS * 32)
k_export_rows_idx(int64_t n, int n_elem, int stride, const int32_t* __restrict__ perm,
                  const int32_t* __restrict__ nbr, const int32_t* __restrict__ nbr_cnt,
                  const int64_t* __restrict__ offsets, int32_t* __restrict__ idx, int64_t cap) {
    __shared__ int32_t buf[EXP_WARPS][256];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t p = (int64_t)blockIdx.x * EXP_WARPS + wid;
    if (p >= n) return;
    int c = 0;
    for (int e = 0; e < n_elem; ++e) c += nbr_cnt[(size_t)p * MAX_ELEM + e];
    int32_t* b = buf[wid];
    for (int m = lane; m < 256; m += 32) b[m] = m < c ? perm[nbr[(size_t)p * stride + m]] : 0x7fffffff;
    __syncwarp();
    for (int k = 2; k <= 256; k <<= 1)
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int t = lane; t < 256; t += 32) {
                const int x = t ^ j;
                if (x > t) {
                    const int32_t v0 = b[t], v1 = b[x];
                    const bool up = (t & k) == 0;
                    if ((v0 > v1) == up) { b[t] = v1; b[x] = v0; }
                }
            }
            __syncwarp();
        }
    const int64_t o = offsets[perm[p]];
    for (int m = lane; m < c; m += 32)
        if (o + m < cap) idx[o + m] = b[m];
}

int launch_export_neighbors(const Workspace& w, int64_t n, int n_elem, int stride, const int64_t* d_offsets,
                            int32_t* d_idx, int64_t cap, cudaStream_t st) {
    if (n == 0) return 0;
    k_export_rows_idx<<<(unsigned)((n + EXP_WARPS - 1) / EXP_WARPS), EXP_WARPS * 32, 0, st>>>(
        n, n_elem, stride, w.perm, w.nbr, w.nbr_cnt, d_offsets, d_idx, cap);
    return 1;
}

__global__ void k_export_rows(int64_t n, int gs, const int32_t* __restrict__ perm, const double* __restrict__ src,
                              double* __restrict__ dst) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n * gs) return;
    const int64_t p = t / gs;
    const int s = (int)(t - p * gs);
    dst[(size_t)perm[p] * gs + s] = src[t];
}

int launch_export_rows(const Workspace& w, int64_t n, int g_stride, const double* src_sorted, double* dst,
                       cudaStream_t st) {
    if (n == 0) return 0;
    const int64_t tot = n * g_stride;
    k_export_rows<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(n, g_stride, w.perm, src_sorted, dst);
    return 1;
}

// ---------------------------------------------------------------- FP64 issue-rate probe
// 8 independent DFMA chains per thread, enough warps on every SM to saturate the FP64 pipe.
constexpr int PEAK_ITERS = 4096;
constexpr int PEAK_CHAINS = 8;

__global__ void __launch_bounds__(256) k_fp64_peak(double* out, double a, double b) {
    double x[PEAK_CHAINS];
#pragma unroll
    for (int c = 0; c < PEAK_CHAINS; ++c) x[c] = a + c + threadIdx.x * 1e-9;
    for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
        for (int c = 0; c < PEAK_CHAINS; ++c) x[c] = fma(x[c], b, a);
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < PEAK_CHAINS; ++c) s += x[c];
    if (s == 123.456) out[0] = s;   // never true; keeps the chains alive
}

double fp64_peak(int device, double seconds, double* sustained, cudaError_t* err) {
    *err = cudaSetDevice(device);
    if (*err != cudaSuccess) return 0.0;
    cudaDeviceProp prop;
    *err = cudaGetDeviceProperties(&prop, device);
    if (*err != cudaSuccess) return 0.0;
    double* d_out = nullptr;
    *err = cudaMalloc(&d_out, sizeof(double));
    if (*err != cudaSuccess) return 0.0;
    const int blocks = prop.multiProcessorCount * 8;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    for (int w = 0; w < 3; ++w) k_fp64_peak<<<blocks, 256>>>(d_out, 1.0, 0.999999);
    cudaDeviceSynchronize();
    double best = 0.0, elapsed = 0.0, work = 0.0;
    int reps = 0;
    while (elapsed < seconds && reps < 10000) {
        cudaEventRecord(e0);
        for (int r = 0; r < 10; ++r) k_fp64_peak<<<blocks, 256>>>(d_out, 1.0, 0.999999);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double rate = 10.0 * blocks * 256.0 * PEAK_ITERS * PEAK_CHAINS / (ms * 1e-3);
        if (rate > best) best = rate;
        work += 10.0 * blocks * 256.0 * PEAK_ITERS * PEAK_CHAINS;
        elapsed += ms * 1e-3;
        ++reps;
    }
    *err = cudaGetLastError();
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d_out);
    if (sustained) *sustained = elapsed > 0.0 ? work / elapsed : 0.0;
    return best;
}

}  // namespace nnp
