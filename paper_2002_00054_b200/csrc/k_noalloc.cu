// k_noalloc.cu -- the kinetic energy of the MD loop ("energy conservation") for callers
// that cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// nnp_md_kinetic_energy (k_md.cu) writes the block sums of  sum_i m_i |v_i|^2  into the caller's workspace, which
// somebody had to cudaMalloc.  The variant here keeps those block sums in a file-scope device array instead:
//
//     static __device__ __align__(256) double g_ekin_part[NOALLOC_MAX_PARTIALS]      (128 KB)
//
// Every GPU that loads the library holds the array until the process exits.  The launcher below calls no cudaMalloc,
// cudaFree or allocating library routine.  In HOST code the name g_ekin_part is a host-side stand-in, not a device
// address, so the address handed to the kernels comes from cudaGetSymbolAddress, fetched once per device with that
// device current (noalloc_scratch).
//
// Every call on a device shares the array and finds the previous call's contents in it.  Nothing has to start at zero:
// a call overwrites partials [0, nb) and its final kernel reads exactly [0, nb).  Two calls that OVERLAP on the GPU
// (different streams, no ordering between them) race on the array -- keep the calls on one stream, or order them.
//
// Arithmetic and summation order are those of k_ekin_partial / k_ekin_final in k_md.cu (256-thread tree per block,
// then the partials in a fixed order), so the result has the same bits as nnp_md_kinetic_energy's.
#include "nnp_internal.h"

namespace nnp {

static __device__ __align__(256) double g_ekin_part[NOALLOC_MAX_PARTIALS];

struct NoallocMass {
    double mass[MAX_ELEM];
};

// block partials of sum m v^2 (fixed order inside the block)
__global__ void __launch_bounds__(256)
k_ekin_partial_static(int64_t n, const int32_t* __restrict__ type, const double* __restrict__ vel, NoallocMass mm,
                      double* __restrict__ part) {
    __shared__ double sh[256];
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    double e = 0.0;
    if (i < n) {
        const double vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
        e = mm.mass[type[i]] * fma(vx, vx, fma(vy, vy, vz * vz));
    }
    sh[threadIdx.x] = e;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) part[blockIdx.x] = sh[0];
}

// one block adds the partials in a fixed order
__global__ void __launch_bounds__(1024)
k_ekin_final_static(int64_t nb, const double* __restrict__ part, double scale, double* __restrict__ out) {
    __shared__ double sh[1024];
    double e = 0.0;
    for (int64_t b = threadIdx.x; b < nb; b += 1024) e += part[b];
    sh[threadIdx.x] = e;
    __syncthreads();
    for (int s = 512; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[0] = scale * sh[0];
}

// Device address of g_ekin_part on the CURRENT device (the caller has made the model's device current).  Looked up
// once per device; a failed lookup is not cached and is returned to the caller.
static cudaError_t noalloc_scratch(double** out) {
    static double* addr[64] = {nullptr};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < 64 && addr[dev]) {
        *out = addr[dev];
        return cudaSuccess;
    }
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_ekin_part);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    if (dev >= 0 && dev < 64) addr[dev] = p;
    *out = p;
    return cudaSuccess;
}

// Enqueues the two kernels on `st`.  n <= NOALLOC_MAX_ATOMS is checked by the caller (nnp_md_kinetic_energy_noalloc).
cudaError_t launch_ekin_noalloc(int64_t n, int n_elem, const double* h_mass, const int32_t* d_type, const double* d_vel,
                                double* d_out, cudaStream_t st, int* launches) {
    double* part = nullptr;
    cudaError_t e = noalloc_scratch(&part);
    if (e != cudaSuccess) return e;
    NoallocMass mm;
    for (int q = 0; q < MAX_ELEM; ++q) mm.mass[q] = q < n_elem ? h_mass[q] : 1.0;
    const int64_t nb = (n + 255) / 256;
    *launches = 0;
    if (n > 0) {
        k_ekin_partial_static<<<(unsigned)nb, 256, 0, st>>>(n, d_type, d_vel, mm, part);
        ++*launches;
    }
    k_ekin_final_static<<<1, 1024, 0, st>>>(n > 0 ? nb : 0, part, 0.5 / NNP_ACC_UNIT, d_out);
    ++*launches;
    return cudaGetLastError();
}

}  // namespace nnp
