// k_mlp.cu -- S3: per-element atomic networks, forward and backward in one kernel
// (PAPER.md L40 step 2: "matrix multiplications that forward-propagate the computed symmetry
// functions ... to calculate the atomic energy"; step 3 needs "the gradient of the neural
// network (w.r.t descriptors)").  E_i = NN_t(G_i), beta_i = dE_i/dG_i.
//   hidden: h = softplus(W h_prev + b) = max(x,0) + log1p(exp(-|x|)),  softplus' = 1/(1+exp(-x));
//   output layer linear (readings 5, C12).
//
// Two kernels: k_mlp_reg (below) for small networks -- n_in -> n1 -> n2 -> 1 with n1, n2 <= 32, the paper's
// "~30 x 2" (L40) and BASELINE.json's 25-25 -- with the weights in the kernel parameter block, and the tiled
// k_mlp<TA> for everything else (the 64-64 networks of the wide config, other depths).
// The paper calls this "a minor portion of the overall computation" (L40, L90); here it is ~1 %
// (base) to ~3 % (wide) of the FP64 work, so it runs on plain DFMA: a tile of TA atoms per CTA,
// activations in shared memory as [neuron][atom] (conflict-free, stride TA+1), each thread owns
// one atom and blocks of 4 output neurons, weights come as 128-bit broadcast loads through L1.
// No tensor cores: B200's FP64 tensor rate equals its FP64 vector rate and the contraction is
// 1-3 % of the step.
#include "mathfn.cuh"
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

// softplus(x) = max(x, 0) + log1p(e) and softplus'(x) = 1 / (1 + exp(-x)) from ONE exponential e = exp(-|x|):
//   u = 1 + e in [1, 2];  sigmoid = (x >= 0 ? 1 : e) / u;
//   log1p(e) = log(u) - ((u - 1) - e) / u      (the second term undoes the rounding of 1 + e: exact to first order, and
//                                               it IS the result once e < 2^-53)
//   log(u) = k ln2 + 2 s P(s^2),  m = u / 2^k in [1/sqrt2, sqrt2],  s = (m - 1) / (m + 1),  P = ATHC (mathfn.cuh, 3e-18).
// libdevice's exp + exp + log1p + division were ~150 FP64-pipe instructions per hidden neuron -- more than the
// network's matrix products; this is ~65 (k_mlp_reg 3.10 -> 2.77 ms at 2.1 M atoms, 1.45 -> 1.23 ms on the Ni-like workload).
__device__ __forceinline__ void softplus_sigmoid(double x, double& h, double& dh) {
    const double e = exp_small(fmax(-fabs(x), -700.0));
    const double u = 1.0 + e;
    const double ru = 1.0 / u;
    const bool big = u > 1.4142135623730951;
    const double m = big ? 0.5 * u : u;
    const double s = (m - 1.0) / (m + 1.0);
    const double q = s * s;
    double p = ATHC[7];
#pragma unroll
    for (int k = 6; k >= 0; --k) p = fma(p, q, ATHC[k]);
    double lg = (s + s) * p;
    if (big) lg += 0.69314718055994531;
    const double l1p = fma(-((u - 1.0) - e), ru, lg);
    h = fmax(x, 0.0) + l1p;
    dh = x >= 0.0 ? ru : e * ru;
}
// hidden activation and its derivative: kind 0 softplus (BASELINE.json), 1 tanh
__device__ __forceinline__ void activate(int kind, double z, double& h, double& dh) {
    if (kind == 1) { h = tanh(z); dh = fma(-h, h, 1.0); }
    else softplus_sigmoid(z, h, dh);
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

// ---- register kernel for small networks (n_in -> n1 -> n2 -> 1, n1, n2 <= 32, n_in <= 80) ----------------
// One thread per atom, every activation in registers, the weights in the kernel PARAMETER block: their
// index is warp-uniform, so they arrive through the constant cache in uniform registers (LDCU) and the
// FP64 FMAs take them as operands -- no shared-memory or L1 operand traffic at all.  The tiled kernel above
// is bound by exactly that traffic (3 loads per 4 FMAs): 4.6 ms at 2.1 M atoms against ~1 ms of FP64 work.
struct MlpRegParams {
    MlpRegWeights W;
    const int32_t* elem_begin;
    const int32_t* elem_end;
    const double* G;
    double* dEdG;
    double* e_sorted;
    const double* sf_shift;
    const double* sf_scale;
    int g_stride, activation;
};
static_assert(sizeof(MlpRegParams) <= 32000, "kernel parameter block limit (32,764 B)");

constexpr int MLP_REG_THREADS = 64;

// Loops are ROLLED over the input index (run-time, warp-uniform -> LDCU weight loads) and UNROLLED over the
// 32 outputs held in registers; per-thread hidden activations / derivatives sit in shared memory as
// [neuron][thread] columns (conflict-free), so no register array is ever indexed dynamically.
__global__ void __launch_bounds__(MLP_REG_THREADS) k_mlp_reg(const __grid_constant__ MlpRegParams p) {
    constexpr int H = MLP_REG_H, NT = MLP_REG_THREADS;
    // only the rows the network has (25 + 25 of 64 for BASELINE.json's): shared memory bounds the resident CTAs (ncu: 6 of 64-row
    // CTAs per SM, 19 % of the warp slots)
    extern __shared__ __align__(16) double sm_reg[];
    const int nh = p.W.n1 > p.W.n2 ? p.W.n1 : p.W.n2;
    double (*sh_h)[NT] = reinterpret_cast<double (*)[NT]>(sm_reg);               // [nh]: h1, later z2 / delta_2, delta_1
    double (*sh_s)[NT] = reinterpret_cast<double (*)[NT]>(sm_reg) + nh;          // [n1]: act'(z1)
    const int t = threadIdx.x;
    const int begin = *p.elem_begin, end = *p.elem_end;
    const int64_t a = (int64_t)begin + (int64_t)blockIdx.x * NT + t;
    if (a >= end) return;                        // no barrier below: a thread only touches its own column
    const int n_in = p.W.n_in, n1 = p.W.n1, n2 = p.W.n2, gs = p.g_stride;
    const double* W1 = p.W.w;                    // [n_in][H]
    const double* B1 = W1 + n_in * H;
    const double* W2 = B1 + H;                   // [H][H], input-major
    const double* B2 = W2 + H * H;
    const double* W3 = B2 + H;
    const double* Grow = p.G + (size_t)a * gs;
    double* Brow = p.dEdG + (size_t)a * gs;

    double acc[H];
    // ---- forward, layer 1: z1 = b1 + W1^T x
#pragma unroll
    for (int o = 0; o < H; ++o) acc[o] = B1[o];
#pragma unroll 1
    for (int i = 0; i < n_in; ++i) {
        double x = Grow[i];
        if (p.sf_scale) x = p.sf_scale[i] * (x - p.sf_shift[i]);
#pragma unroll
        for (int o = 0; o < H; ++o) acc[o] = fma(W1[i * H + o], x, acc[o]);
    }
#pragma unroll
    for (int o = 0; o < H; ++o)
        if (o < n1) sh_h[o][t] = acc[o];
#pragma unroll 1
    for (int o = 0; o < n1; ++o) {               // rolled: ONE copy of the activation code
        double h, d;
        activate(p.activation, sh_h[o][t], h, d);
        sh_h[o][t] = h;
        sh_s[o][t] = d;
    }
    // ---- layer 2: z2 = b2 + W2^T h1
#pragma unroll
    for (int o = 0; o < H; ++o) acc[o] = B2[o];
#pragma unroll 1
    for (int i = 0; i < n1; ++i) {
        const double x = sh_h[i][t];
#pragma unroll
        for (int o = 0; o < H; ++o) acc[o] = fma(W2[i * H + o], x, acc[o]);
    }
    double e = W3[H];                            // b3
#pragma unroll
    for (int o = 0; o < H; ++o)
        if (o < n2) sh_h[o][t] = acc[o];         // h1 is dead: its columns take z2, then delta_2
#pragma unroll 1
    for (int o = 0; o < n2; ++o) {
        double h, d;
        activate(p.activation, sh_h[o][t], h, d);
        e = fma(W3[o], h, e);
        sh_h[o][t] = W3[o] * d;                  // delta_2[o] = w3[o] act'(z2[o])
    }
#pragma unroll
    for (int o = 0; o < H; ++o) acc[o] = o < n2 ? sh_h[o][t] : 0.0;
    p.e_sorted[a] = e;
    // ---- backward: delta_1[i] = act'(z1[i]) sum_o W2[i][o] delta_2[o]   (delta_2 in registers)
#pragma unroll 1
    for (int i = 0; i < n1; ++i) {
        double g0 = 0.0, g1 = 0.0, g2 = 0.0, g3 = 0.0;
#pragma unroll
        for (int o = 0; o < H; o += 4) {
            g0 = fma(W2[i * H + o], acc[o], g0);
            g1 = fma(W2[i * H + o + 1], acc[o + 1], g1);
            g2 = fma(W2[i * H + o + 2], acc[o + 2], g2);
            g3 = fma(W2[i * H + o + 3], acc[o + 3], g3);
        }
        sh_h[i][t] = sh_s[i][t] * ((g0 + g1) + (g2 + g3));
    }
    // ---- beta_k = dE/dG_k = scale_k sum_i W1[k][i] delta_1[i]   (delta_1 into registers)
#pragma unroll
    for (int i = 0; i < H; ++i) acc[i] = i < n1 ? sh_h[i][t] : 0.0;
#pragma unroll 1
    for (int k = 0; k < n_in; ++k) {
        double g0 = 0.0, g1 = 0.0, g2 = 0.0, g3 = 0.0;
#pragma unroll
        for (int i = 0; i < H; i += 4) {
            g0 = fma(W1[k * H + i], acc[i], g0);
            g1 = fma(W1[k * H + i + 1], acc[i + 1], g1);
            g2 = fma(W1[k * H + i + 2], acc[i + 2], g2);
            g3 = fma(W1[k * H + i + 3], acc[i + 3], g3);
        }
        double b = (g0 + g1) + (g2 + g3);
        if (p.sf_scale) b *= p.sf_scale[k];
        Brow[k] = b;
    }
    for (int k = n_in; k < gs; ++k) Brow[k] = 0.0;
}

size_t mlp_smem_bytes(const NetDesc& net, int TA) {
    size_t rows = net.sizes[0] + 1;
    for (int l = 1; l < net.n_layers; ++l) rows += 2 * (size_t)net.sizes[l];
    return rows * (TA + 1) * sizeof(double);
}

template <int TA>
static void launch_ta(const MlpParams& p, int64_t n, size_t smem, cudaStream_t st) {
    static unsigned long long configured = 0ull;      // per device (opt_in_smem)
    opt_in_smem(k_mlp<TA>, &configured);
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
        if (nets[e].reg) {          // small network: register kernel, weights in the parameter block
            MlpRegParams q;
            q.W = *nets[e].reg;
            q.elem_begin = p.elem_begin; q.elem_end = p.elem_end;
            q.G = w.G; q.dEdG = w.dEdG; q.e_sorted = w.e_sorted;
            q.sf_shift = nets[e].sf_shift; q.sf_scale = nets[e].sf_scale;
            q.g_stride = g_stride; q.activation = nets[e].activation;
            const int nh = q.W.n1 > q.W.n2 ? q.W.n1 : q.W.n2;
            const size_t smem = (size_t)(nh + q.W.n1) * MLP_REG_THREADS * sizeof(double);      // <= 32 KB
            k_mlp_reg<<<(unsigned)((n + MLP_REG_THREADS - 1) / MLP_REG_THREADS), MLP_REG_THREADS, smem, st>>>(q);
            ++launches;
            continue;
        }
        // Atoms per CTA: the 256 threads form 256 / TA groups that each own blocks of four outputs, so TA is chosen
        // to give as many groups as the widest hidden layer has blocks -- 25 wide: 7 blocks, 8 groups, 32 atoms
        // (4.6 ms against 6.5 ms with 64 atoms at 2.1 M atoms); 64 wide: 16 blocks, 16 groups, 16 atoms (2.0 ms against
        // 3.2 ms with 32 atoms on configs[4]: half the shared memory per CTA, twice the resident warps)
        int widest = 1;
        for (int l = 1; l < p.net.n_layers; ++l) widest = p.net.sizes[l] > widest ? p.net.sizes[l] : widest;
        const int blocks = (widest + 3) / 4;
        const size_t budget = 100 * 1024;
        if (blocks <= 8 && mlp_smem_bytes(p.net, 32) <= budget) launch_ta<32>(p, n, mlp_smem_bytes(p.net, 32), st);
        else if (blocks <= 16 && mlp_smem_bytes(p.net, 16) <= 2 * budget) launch_ta<16>(p, n, mlp_smem_bytes(p.net, 16), st);
        else launch_ta<8>(p, n, mlp_smem_bytes(p.net, 8), st);
        ++launches;
    }
    return launches;
}

}  // namespace nnp
