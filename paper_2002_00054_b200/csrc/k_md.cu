// k_md.cu -- the MD loop around the path ("energy conservation"):
// velocity-Verlet NVE on the device.  HBM-bound elementwise kernels (72 B read + 48 B written per atom
// for kick+drift); against the ~140 ms force evaluation they are noise, so they are kept simple.
#include "nnp_internal.h"

namespace nnp {

struct MdMass {
    double inv_mass[MAX_ELEM];   // NNP_ACC_UNIT / m_e
    double mass[MAX_ELEM];
};

// v += hdt * F/m (acceleration unit folded into inv_mass); optionally x += dt * v
__global__ void __launch_bounds__(256)
k_vv_kick_drift(int64_t n3, const int32_t* __restrict__ type, const double* __restrict__ force, double* __restrict__ vel,
                double* __restrict__ pos, MdMass mm, double hdt, double dt, int drift) {
    const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n3) return;
    const int t = type[q / 3];
    const double v = fma(hdt * mm.inv_mass[t], force[q], vel[q]);
    vel[q] = v;
    if (drift) pos[q] = fma(dt, v, pos[q]);
}

// block partials of sum m v^2 (fixed order inside the block), then one block adds the partials in order
__global__ void __launch_bounds__(256)
k_ekin_partial(int64_t n, const int32_t* __restrict__ type, const double* __restrict__ vel, MdMass mm, double* __restrict__ part) {
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

__global__ void __launch_bounds__(1024) k_ekin_final(int64_t nb, const double* __restrict__ part, double scale, double* out) {
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

static MdMass make_mass(const double* h_mass, int n_elem) {
    MdMass mm;
    for (int e = 0; e < MAX_ELEM; ++e) {
        mm.mass[e] = e < n_elem ? h_mass[e] : 1.0;
        mm.inv_mass[e] = NNP_ACC_UNIT / mm.mass[e];
    }
    return mm;
}

int launch_vv(int64_t n, int n_elem, const double* h_mass, const int32_t* d_type, const double* d_force, double* d_vel,
              double* d_pos, double dt, bool drift, cudaStream_t st) {
    if (n == 0) return 0;
    const int64_t n3 = 3 * n;
    k_vv_kick_drift<<<(unsigned)((n3 + 255) / 256), 256, 0, st>>>(n3, d_type, d_force, d_vel, d_pos, make_mass(h_mass, n_elem),
                                                                  0.5 * dt, dt, drift ? 1 : 0);
    return 1;
}

int launch_ekin(int64_t n, int n_elem, const double* h_mass, const int32_t* d_type, const double* d_vel, double* d_part,
                double* d_out, cudaStream_t st) {
    const int64_t nb = (n + 255) / 256;
    if (n > 0) k_ekin_partial<<<(unsigned)nb, 256, 0, st>>>(n, d_type, d_vel, make_mass(h_mass, n_elem), d_part);
    k_ekin_final<<<1, 1024, 0, st>>>(n > 0 ? nb : 0, d_part, 0.5 / NNP_ACC_UNIT, d_out);
    return 2;
}

}  // namespace nnp
