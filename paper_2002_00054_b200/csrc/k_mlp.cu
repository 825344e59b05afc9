// k_mlp.cu -- S3: per-element atomic networks, forward and backward in one kernel
// (PAPER.md L40 step 2: "matrix multiplications that forward-propagate the computed symmetry
// functions ... to calculate the atomic energy"; step 3 needs "the gradient of the neural
// network (w.r.t descriptors)").  E_i = NN_t(G_i), beta_i = dE_i/dG_i.
//   hidden: h = softplus(W h_prev + b) = max(x,0) + log1p(exp(-|x|)),  softplus' = 1/(1+exp(-x));
//   output layer linear (readings 5, C12).
//
// The paper calls this "a minor portion of the overall computation" (L40, L90); here it is ~1 %
// (base) to ~3 % (wide) of the FP64 work, so it runs on plain DFMA: a tile of TA atoms per CTA,
// activations in shared memory as [neuron][atom] (conflict-free, stride TA+1), each thread owns
// one atom and blocks of 4 output neurons, weights come as 128-bit broadcast loads through L1.
// No tensor cores: B200's FP64 tensor rate equals its FP64 vector rate and the contraction is
// 1-3 % of the step.
#include "nnp_internal.h"

namespace nnp {

constexpr int MLP_THREADS = 256;

struct MlpParams {
    NetDesc net;
    const int32_t* elem_begin;   // device: first sorted index of this element
    const int32_t* elem_end;     // device: one past the last
    const double* G;
    double* dEdG;
    double* e_sorted;
    int g_stride;
};

__device__ __forceinline__ double softplus_d(double x) { return fmax(x, 0.0) + log1p(exp(-fabs(x))); }
__device__ __forceinline__ double sigmoid_d(double x) { return 1.0 / (1.0 + exp(-x)); }
// hidden activation and its derivative: kind 0 softplus (BASELINE.json), 1 tanh
__device__ __forceinline__ void activate(int kind, double z, double& h, double& dh) {
    if (kind == 1) { h = tanh(z); dh = fma(-h, h, 1.0); }
    else { h = softplus_d(z); dh = sigmoid_d(z); }
}

__host__ __device__ inline int round4(int x) { return (x + 3) & ~3; }

template <int TA>
__global__ void __launch_bounds__(MLP_THREADS) k_mlp(const __grid_constant__ MlpParams p) {
    constexpr int TAP = TA + 1;
    constexpr int NG = MLP_THREADS / TA;
    extern __shared__ __align__(16) double sm[];
    const int begin = *p.elem_begin, end = *p.elem_end;
    const int64_t start = (int64_t)begin + (int64_t)blockIdx.x * TA;
    if (start >= end) return;
    const int na = (int)min((int64_t)TA, (int64_t)end - start);
    const int t = threadIdx.x, a = t % TA, grp = t / TA;
    const NetDesc& net = p.net;
    const int L = net.n_layers, n_in = net.sizes[0], gs = p.g_stride;

    // shared-memory map: X0 [n_in][TAP]; for hidden layer l=1..L-1: A_l, D_l [sizes[l]][TAP]; top [TAP]
    double* X0 = sm;
    double* Al[MAX_LAYERS + 1];
    double* Dl[MAX_LAYERS + 1];
    {
        double* q = X0 + (size_t)n_in * TAP;
        for (int l = 1; l < L; ++l) {
            Al[l] = q; q += (size_t)net.sizes[l] * TAP;
            Dl[l] = q; q += (size_t)net.sizes[l] * TAP;
        }
        Al[L] = q;   // "top": dE/dE = 1
        Al[0] = X0;
    }

    for (int idx = t; idx < TA * n_in; idx += MLP_THREADS) {
        const int aa = idx / n_in, s = idx - aa * n_in;
        double x = aa < na ? p.G[(size_t)(start + aa) * gs + s] : 0.0;
        if (net.sf_scale) x = net.sf_scale[s] * (x - net.sf_shift[s]);      // affine SF scaling (8(f)4)
        X0[s * TAP + aa] = x;
    }
    if (t < TA) Al[L][t] = 1.0;
    __syncthreads();

    // ---- forward ---------------------------------------------------------------------------
    for (int l = 0; l < L; ++l) {
        const int nin = net.sizes[l], nout = net.sizes[l + 1], np = round4(nout);
        const double* __restrict__ WT = net.weights + net.wt_off[l];   // [nin][np]
        const double* __restrict__ B = net.weights + net.b_off[l];     // [np]
        const double* in = Al[l];
        for (int ob = grp * 4; ob < nout; ob += NG * 4) {
            const double2 b01 = __ldg(reinterpret_cast<const double2*>(B + ob));
            const double2 b23 = __ldg(reinterpret_cast<const double2*>(B + ob + 2));
            double z0 = b01.x, z1 = b01.y, z2 = b23.x, z3 = b23.y;
            for (int i = 0; i < nin; ++i) {
                const double x = in[i * TAP + a];
                const double2 w01 = __ldg(reinterpret_cast<const double2*>(WT + (size_t)i * np + ob));
                const double2 w23 = __ldg(reinterpret_cast<const double2*>(WT + (size_t)i * np + ob + 2));
                z0 = fma(w01.x, x, z0); z1 = fma(w01.y, x, z1);
                z2 = fma(w23.x, x, z2); z3 = fma(w23.y, x, z3);
            }
            const double z[4] = {z0, z1, z2, z3};
            if (l < L - 1) {
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (ob + k < nout) {
                        double h, dh;
                        activate(net.activation, z[k], h, dh);
                        Al[l + 1][(ob + k) * TAP + a] = h;
                        Dl[l + 1][(ob + k) * TAP + a] = dh;
                    }
            } else if (ob == 0 && a < na) {
                p.e_sorted[start + a] = z0;
            }
        }
        __syncthreads();
    }

    // ---- backward: delta_L = 1; g_in = W^T delta; delta_l = g_in * softplus'(z_l) ---------------
    for (int l = L - 1; l >= 0; --l) {
        const int nin = net.sizes[l], nout = net.sizes[l + 1], npi = round4(nin);
        const double* __restrict__ W = net.weights + net.w_off[l];   // [nout][npi]
        const double* delta = Al[l + 1];
        for (int ib = grp * 4; ib < nin; ib += NG * 4) {
            double g0 = 0.0, g1 = 0.0, g2 = 0.0, g3 = 0.0;
            for (int o = 0; o < nout; ++o) {
                const double d = delta[o * TAP + a];
                const double2 w01 = __ldg(reinterpret_cast<const double2*>(W + (size_t)o * npi + ib));
                const double2 w23 = __ldg(reinterpret_cast<const double2*>(W + (size_t)o * npi + ib + 2));
                g0 = fma(w01.x, d, g0); g1 = fma(w01.y, d, g1);
                g2 = fma(w23.x, d, g2); g3 = fma(w23.y, d, g3);
            }
            const double g[4] = {g0, g1, g2, g3};
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (ib + k < nin) {
                    const int q = (ib + k) * TAP + a;
                    Al[l][q] = l > 0 ? g[k] * Dl[l][q] : g[k];
                }
        }
        __syncthreads();
    }

    for (int idx = t; idx < na * gs; idx += MLP_THREADS) {
        const int aa = idx / gs, s = idx - aa * gs;
        double b = s < n_in ? X0[s * TAP + aa] : 0.0;
        if (net.sf_scale && s < n_in) b *= net.sf_scale[s];                 // dE/dG = scale * dE/dx
        p.dEdG[(size_t)(start + aa) * gs + s] = b;
    }
}

size_t mlp_smem_bytes(const NetDesc& net, int TA) {
    size_t rows = net.sizes[0] + 1;
    for (int l = 1; l < net.n_layers; ++l) rows += 2 * (size_t)net.sizes[l];
    return rows * (TA + 1) * sizeof(double);
}

template <int TA>
static void launch_ta(const MlpParams& p, int64_t n, size_t smem, cudaStream_t st) {
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(k_mlp<TA>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        configured = true;
    }
    const unsigned nb = (unsigned)((n + TA - 1) / TA);   // upper bound; CTAs past the element's range exit
    k_mlp<TA><<<nb, MLP_THREADS, smem, st>>>(p);
}

int launch_mlp(const Workspace& w, int64_t n, int n_elem, int ncell, const NetDesc* nets, int g_stride,
               cudaStream_t st) {
    if (n == 0) return 0;
    int launches = 0;
    for (int e = 0; e < n_elem; ++e) {
        MlpParams p;
        p.net = nets[e];
        p.elem_begin = w.cell_start + (size_t)e * ncell;
        p.elem_end = w.cell_start + (size_t)(e + 1) * ncell;
        p.G = w.G; p.dEdG = w.dEdG; p.e_sorted = w.e_sorted; p.g_stride = g_stride;
        const size_t budget = 100 * 1024;
        // 32 atoms per CTA: 8 thread groups cover the 7 output blocks of a 25-wide layer in one round
        // (measured 4.6 ms against 6.5 ms with 64 atoms / 4 groups at 2.1 M atoms)
        if (mlp_smem_bytes(p.net, 32) <= budget) launch_ta<32>(p, n, mlp_smem_bytes(p.net, 32), st);
        else if (mlp_smem_bytes(p.net, 16) <= 2 * budget) launch_ta<16>(p, n, mlp_smem_bytes(p.net, 16), st);
        else launch_ta<8>(p, n, mlp_smem_bytes(p.net, 8), st);
        ++launches;
    }
    return launches;
}

}  // namespace nnp
