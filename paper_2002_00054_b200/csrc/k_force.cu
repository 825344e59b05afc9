// k_force.cu -- S4: forces  F_m = - sum_i sum_s beta_is dG_is/dr_m  with beta = dE_i/dG_i from the
// network kernel and dG/dr RECOMPUTED here, never stored (PAPER.md L40 step 3, L56-58 "store and
// move as little data as possible, recomputing where necessary", L98, L124).  This holds "the
// dominant angular force loop" (L116) and is the hottest kernel of the path.
//
// One warp per centre i, same staging / tournament enumeration / compaction as k_sf.cu.  For a
// triplet (i; j,k) with u = r_j - r_i, v = r_k - r_i, w = v - u the beta-weighted gradient is
//     dg/du = f_uu u + f_uv v - f_w w,      dg/dv = f_vv v + f_uv u + f_w w
// (DESIGN.md "Force algebra"); the forces on j and k are accumulated per neighbour SLOT in shared
// memory (FP64 atomicAdd = CAS loop; the tournament order keeps same-address collisions inside a
// batch to <= 2-3), and each slot is flushed ONCE per centre with global FP64 atomics.
#include "angular.cuh"
#include "geometry.cuh"

namespace nnp {

constexpr int FC_WARPS = 4;
constexpr double PI_D = 3.14159265358979323846;

struct ForceParams {
    int64_t n;
    int n_elem, ncell, stride, cap, g_stride;
    double rc, rc2, inv_rc;
    double box[3], half[3];
    const double *sx, *sy, *sz;
    const int32_t *cell_start, *nbr, *nbr_cnt;
    const double* dEdG;
    double* f_sorted;
    const ElemProgram* prog[MAX_ELEM];
    int variant[MAX_ELEM];
};

template <class Spec>
__host__ __device__ constexpr size_t force_warp_smem(int cap, int g_stride) {
    // p0,p1,p2 + pe per slot + slot forces (3 doubles) ; queue ; beta row ; per-group coefficient tables
    size_t b = (size_t)cap * (48 + 8 * Spec::NETA + 24) + 128 + (size_t)g_stride * 8;
    b += (size_t)2 * Spec::NACC * 8;
    return (b + 15) / 16 * 16;
}

// shared "slot force" accumulators
struct SlotF {
    double *x, *y, *z;
};

// common tail of the per-triplet work: from Z0 = sum beta P Y, Z1 = sum beta P' Y, Z2 = sum eta beta P Y
// (Y = product of the three bare Gaussians) to the two slot forces.
__device__ __forceinline__ void triplet_forces(const double2 j0, const double2 j1, const double2 j2, const double2 k0,
                                               const double2 k1, const double2 k2, double fcc, double dfc, double cosv,
                                               double Z0, double Z1, double Z2, const SlotF& sf, int j, int k, bool active) {
    const double fa = j2.x, dfa = j2.y, fb = k2.x, dfb = k2.y, ia = j1.y, ib = k1.y;
    const double fab = fa * fb;
    const double C = fab * fcc;
    const double t2 = 2.0 * C * Z2;
    const double f_w = (fab * dfc) * Z0 - t2;
    const double q = Z1 * C;
    const double qc = q * cosv;
    const double f_uu = (dfa * fb * fcc) * Z0 - t2 - qc * (ia * ia);
    const double f_vv = (fa * dfb * fcc) * Z0 - t2 - qc * (ib * ib);
    const double f_uv = q * (ia * ib);
    const double s1 = f_uu + f_w, s2 = f_vv + f_w, s3 = f_w - f_uv;
    // F_j = -dg/du = -s1 u + s3 v ;  F_k = -dg/dv = -s2 v + s3 u
    if (!active) return;
    atomicAdd(&sf.x[j], s3 * k0.x - s1 * j0.x);
    atomicAdd(&sf.y[j], s3 * k0.y - s1 * j0.y);
    atomicAdd(&sf.z[j], s3 * k1.x - s1 * j1.x);
    atomicAdd(&sf.x[k], s3 * j0.x - s2 * k0.x);
    atomicAdd(&sf.y[k], s3 * j0.y - s2 * k0.y);
    atomicAdd(&sf.z[k], s3 * j1.x - s2 * k1.x);
}

template <class Spec>
struct ForceTripletFast {
    const Nbh& nb;
    SlotF sf;
    const double* bt0;   // [NACC] beta * 2^(1-zeta)                      (this group)
    const double* bt1;   // [NACC] beta * 2^(1-zeta) * zeta * lambda
    double etas[Spec::NETA > 0 ? Spec::NETA : 1];
    double inv_rc;

    __device__ __forceinline__ void operator()(int j, int k, bool active) {
        const double2 j0 = nb.p0[j], j1 = nb.p1[j], j2 = nb.p2[j];
        const double2 k0 = nb.p0[k], k1 = nb.p1[k], k2 = nb.p2[k];
        const double wx = k0.x - j0.x, wy = k0.y - j0.y, wz = k1.x - j1.x;
        const double c2 = wx * wx + wy * wy + wz * wz;
        const double ic = rsqrt(c2);
        const double c = c2 * ic;
        double sn, cs;
        sincospi(c * inv_rc, &sn, &cs);
        double fcc = 0.5 * cs + 0.5;
        double dfc = (-0.5 * PI_D * inv_rc) * sn * ic;          // fc'(c)/c
        if (!active) { fcc = 0.0; dfc = 0.0; }
        double Ec[Spec::NETA];
        eta_chain<Spec>(c2, etas[0], Ec);
        const double cosv = (j0.x * k0.x + j0.y * k0.y + j1.x * k1.x) * (j1.y * k1.y);
        // pw[l][b] = (1 +- cos)^(2^b) ; pd[l][b] = (1 +- cos)^(2^b - 1)
        double pw[2][Spec::MAXBIT + 1], pd[2][Spec::MAXBIT + 1];
        pw[0][0] = 1.0 + cosv; pw[1][0] = 1.0 - cosv;
        pd[0][0] = 1.0; pd[1][0] = 1.0;
#pragma unroll
        for (int b = 1; b <= Spec::MAXBIT; ++b) {
#pragma unroll
            for (int l = 0; l < 2; ++l) {
                pw[l][b] = pw[l][b - 1] * pw[l][b - 1];
                pd[l][b] = pd[l][b - 1] * pw[l][b - 1];
            }
        }
        double Z0 = 0.0, Z1 = 0.0, Z2 = 0.0;
#pragma unroll
        for (int e = 0; e < Spec::NETA; ++e) {
            double T0 = 0.0, T1 = 0.0;
#pragma unroll
            for (int b = 0; b <= Spec::MAXBIT; ++b) {
#pragma unroll
                for (int l = 0; l < 2; ++l)
                    if (Spec::mask(e) >> (8 * l + b) & 1u) {
                        const int a = acc_index<Spec>(e, 8 * l + b);
                        T0 = fma(bt0[a], pw[l][b], T0);
                        T1 = fma(bt1[a], pd[l][b], T1);
                    }
            }
            const double Y = (nb.pe[j * Spec::NETA + e] * nb.pe[k * Spec::NETA + e]) * Ec[e];
            Z0 = fma(T0, Y, Z0);
            Z1 = fma(T1, Y, Z1);
            Z2 = fma(etas[e] * T0, Y, Z2);
        }
        triplet_forces(j0, j1, j2, k0, k1, k2, fcc, dfc, cosv, Z0, Z1, Z2, sf, j, k, active);
    }
};

struct ForceTripletGeneric {
    const Nbh& nb;
    SlotF sf;
    const AngularSF* list;
    int nsf;
    const double* brow;   // beta row of the centre (shared memory)
    double inv_rc;

    __device__ __forceinline__ void operator()(int j, int k, bool active) {
        const double2 j0 = nb.p0[j], j1 = nb.p1[j], j2 = nb.p2[j];
        const double2 k0 = nb.p0[k], k1 = nb.p1[k], k2 = nb.p2[k];
        const double wx = k0.x - j0.x, wy = k0.y - j0.y, wz = k1.x - j1.x;
        const double c2 = wx * wx + wy * wy + wz * wz;
        const double ic = rsqrt(c2);
        const double c = c2 * ic;
        double sn, cs;
        sincospi(c * inv_rc, &sn, &cs);
        double fcc = 0.5 * cs + 0.5;
        double dfc = (-0.5 * PI_D * inv_rc) * sn * ic;
        if (!active) { fcc = 0.0; dfc = 0.0; }
        const double cosv = (j0.x * k0.x + j0.y * k0.y + j1.x * k1.x) * (j1.y * k1.y);
        const double a2 = 1.0 / (j1.y * j1.y), b2 = 1.0 / (k1.y * k1.y);
        const double r2sum = a2 + b2 + c2;
        double Z0 = 0.0, Z1 = 0.0, Z2 = 0.0;
        for (int s = 0; s < nsf; ++s) {
            const AngularSF f = list[s];
            const double base = 1.0 + (double)f.lam * cosv;
            // base^(zeta-1) and base^zeta
            double pd = 1.0, bb = base;
            for (int z = f.izeta - 1; z > 0; z >>= 1) {
                if (z & 1) pd *= bb;
                bb *= bb;
            }
            const double pwv = pd * base;
            const double Y = exp(-f.eta * r2sum);
            const double bc = brow[f.g] * f.coef;
            Z0 = fma(bc * pwv, Y, Z0);
            Z1 = fma(bc * (double)(f.izeta * f.lam) * pd, Y, Z1);
            Z2 = fma(f.eta * bc * pwv, Y, Z2);
        }
        triplet_forces(j0, j1, j2, k0, k1, k2, fcc, dfc, cosv, Z0, Z1, Z2, sf, j, k, active);
    }
};

template <class Spec>
__global__ void __launch_bounds__(FC_WARPS * 32) k_force(const __grid_constant__ ForceParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t i = (int64_t)blockIdx.x * FC_WARPS + wid;
    if (i >= p.n) return;
    int tc = 0;
    for (int e = 1; e < p.n_elem; ++e)
        if (i >= p.cell_start[(size_t)e * p.ncell]) tc = e;
    if (p.variant[tc] != Spec::ID) return;
    const ElemProgram* __restrict__ prog = p.prog[tc];

    unsigned char* base = smem_raw + (size_t)wid * force_warp_smem<Spec>(p.cap, p.g_stride);
    Nbh nb;
    nb.p0 = reinterpret_cast<double2*>(base);
    nb.p1 = nb.p0 + p.cap;
    nb.p2 = nb.p1 + p.cap;
    nb.pe = reinterpret_cast<double*>(nb.p2 + p.cap);
    SlotF sf;
    sf.x = nb.pe + (size_t)p.cap * Spec::NETA;
    sf.y = sf.x + p.cap;
    sf.z = sf.y + p.cap;
    double* brow = sf.z + p.cap;
    double* bt0 = brow + p.g_stride;
    double* bt1 = bt0 + Spec::NACC;
    PairQueue Q;
    Q.q = reinterpret_cast<uint16_t*>(bt1 + Spec::NACC);
    Q.n = 0;

    int seg[MAX_ELEM + 1];
    seg[0] = 0;
#pragma unroll
    for (int e = 0; e < MAX_ELEM; ++e) seg[e + 1] = seg[e] + p.nbr_cnt[(size_t)i * MAX_ELEM + e];
    const int ntot = seg[MAX_ELEM];

    for (int s = lane; s < p.g_stride; s += 32) brow[s] = p.dEdG[(size_t)i * p.g_stride + s];
    __syncwarp();

    // ---- stage the neighbourhood; radial forces go straight into the slot accumulators ----------
    const double xi = p.sx[i], yi = p.sy[i], zi = p.sz[i];
    const int32_t* row = p.nbr + (size_t)i * p.stride;
    double eta0 = 0.0;
    if constexpr (Spec::NETA > 0) eta0 = prog->ang_eta[0];
    for (int e = 0; e < p.n_elem; ++e) {
        const int nr = prog->n_rad[e], off = prog->rad_off[e];
        for (int m = seg[e] + lane; m < seg[e + 1]; m += 32) {
            const int j = row[m];
            const double dx = min_image_1d(xi, p.sx[j], p.box[0], p.half[0]);
            const double dy = min_image_1d(yi, p.sy[j], p.box[1], p.half[1]);
            const double dz = min_image_1d(zi, p.sz[j], p.box[2], p.half[2]);
            const double a2 = dx * dx + dy * dy + dz * dz;
            const double ia = rsqrt(a2);
            const double a = a2 * ia;
            double sn, cs;
            sincospi(a * p.inv_rc, &sn, &cs);
            const double fa = 0.5 * cs + 0.5;
            const double dfa_r = (-0.5 * PI_D * p.inv_rc) * sn;   // fc'(a)
            nb.p0[m] = make_double2(dx, dy);
            nb.p1[m] = make_double2(dz, ia);
            nb.p2[m] = make_double2(fa, dfa_r * ia);
            if constexpr (Spec::NETA > 0) {
                double E[Spec::NETA];
                eta_chain<Spec>(a2, eta0, E);
#pragma unroll
                for (int q = 0; q < Spec::NETA; ++q) nb.pe[m * Spec::NETA + q] = E[q];
            }
            // R = sum_r beta_r exp(-eta d^2) (fc' - 2 eta d fc) / a ;  F_j = -R u
            double R = 0.0;
            for (int r = 0; r < nr; ++r) {
                const RadialSF f = prog->rad[off + r];
                const double d = a - f.rs;
                R = fma(brow[f.g] * exp(-f.eta * d * d), dfa_r - 2.0 * f.eta * d * fa, R);
            }
            R *= ia;
            sf.x[m] = -R * dx;
            sf.y[m] = -R * dy;
            sf.z[m] = -R * dz;
        }
    }
    __syncwarp();

    // ---- angular groups -----------------------------------------------------------------------
    for (int e1 = 0; e1 < p.n_elem; ++e1)
        for (int e2 = e1; e2 < p.n_elem; ++e2) {
            const int pr = pair_index(e1, e2, p.n_elem);
            const int na = prog->n_ang[pr];
            if (na == 0) continue;
            if constexpr (Spec::ID != ANG_GENERIC) {
                // coefficient tables of this group
                if (lane < 16) {
#pragma unroll
                    for (int e = 0; e < Spec::NETA; ++e) {
                        if (Spec::mask(e) >> lane & 1u) {
                            const int g = prog->ang_g[pr][e][lane];
                            const int zeta = 1 << (lane & 7);
                            const double lam = lane < 8 ? 1.0 : -1.0;
                            const double bc = g >= 0 ? brow[g] * exp2((double)(1 - zeta)) : 0.0;
                            int a = 0;   // accumulator slot = set bits before (e, lane)
                            for (int ee = 0; ee < Spec::NETA; ++ee) {
                                const unsigned mk = Spec::mask(ee);
                                if (ee < e) a += __popc(mk);
                                else if (ee == e) a += __popc(mk & ((1u << lane) - 1u));
                            }
                            bt0[a] = bc;
                            bt1[a] = bc * (double)zeta * lam;
                        }
                    }
                }
                __syncwarp();
                ForceTripletFast<Spec> f{nb, sf, bt0, bt1, {}, p.inv_rc};
#pragma unroll
                for (int e = 0; e < Spec::NETA; ++e) f.etas[e] = prog->ang_eta[e];
                if (e1 == e2) enum_within(nb, seg[e1], seg[e1 + 1] - seg[e1], p.rc2, Q, lane, f);
                else enum_between(nb, seg[e1], seg[e1 + 1] - seg[e1], seg[e2], seg[e2 + 1] - seg[e2], p.rc2, Q, lane, f);
                drain_tail(Q, lane, f);
            } else {
                ForceTripletGeneric f{nb, sf, prog->ang + prog->ang_off[pr], na, brow, p.inv_rc};
                if (e1 == e2) enum_within(nb, seg[e1], seg[e1 + 1] - seg[e1], p.rc2, Q, lane, f);
                else enum_between(nb, seg[e1], seg[e1 + 1] - seg[e1], seg[e2], seg[e2 + 1] - seg[e2], p.rc2, Q, lane, f);
                drain_tail(Q, lane, f);
            }
        }
    __syncwarp();

    // ---- flush: one global FP64 atomic per neighbour component; the centre gets minus the sum ----
    double fx = 0.0, fy = 0.0, fz = 0.0;
    for (int m = lane; m < ntot; m += 32) {
        const int j = row[m];
        const double ax = sf.x[m], ay = sf.y[m], az = sf.z[m];
        atomicAdd(&p.f_sorted[3 * (size_t)j + 0], ax);
        atomicAdd(&p.f_sorted[3 * (size_t)j + 1], ay);
        atomicAdd(&p.f_sorted[3 * (size_t)j + 2], az);
        fx -= ax; fy -= ay; fz -= az;
    }
    fx = warp_sum(fx); fy = warp_sum(fy); fz = warp_sum(fz);
    if (lane == 0) {
        atomicAdd(&p.f_sorted[3 * (size_t)i + 0], fx);
        atomicAdd(&p.f_sorted[3 * (size_t)i + 1], fy);
        atomicAdd(&p.f_sorted[3 * (size_t)i + 2], fz);
    }
}

template <class Spec>
static int launch_one(const ForceParams& p, cudaStream_t st) {
    const size_t smem = FC_WARPS * force_warp_smem<Spec>(p.cap, p.g_stride);
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(k_force<Spec>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        configured = true;
    }
    const unsigned nb = (unsigned)((p.n + FC_WARPS - 1) / FC_WARPS);
    k_force<Spec><<<nb, FC_WARPS * 32, smem, st>>>(p);
    return 1;
}

size_t force_smem_bytes(int variant, int cap, int g_stride) {
    switch (variant) {
        case ANG_BASE12: return FC_WARPS * force_warp_smem<SpecBase12>(cap, g_stride);
        case ANG_WIDE32: return FC_WARPS * force_warp_smem<SpecWide32>(cap, g_stride);
        default: return FC_WARPS * force_warp_smem<SpecGeneric>(cap, g_stride);
    }
}

int launch_force(const Workspace& w, const Grid& g, int64_t n, int n_elem, const ElemProgram* const* d_prog,
                 const int* variant, double rc, int stride, int max_nbr, int g_stride, cudaStream_t st) {
    if (n == 0) return 0;
    ForceParams p;
    p.n = n; p.n_elem = n_elem; p.ncell = g.ncell; p.stride = stride; p.cap = max_nbr; p.g_stride = g_stride;
    p.rc = rc; p.rc2 = rc * rc; p.inv_rc = 1.0 / rc;
    for (int c = 0; c < 3; ++c) { p.box[c] = g.box[c]; p.half[c] = g.half[c]; }
    p.sx = w.sx; p.sy = w.sy; p.sz = w.sz;
    p.cell_start = w.cell_start; p.nbr = w.nbr; p.nbr_cnt = w.nbr_cnt; p.dEdG = w.dEdG; p.f_sorted = w.f_sorted;
    bool use[3] = {false, false, false};
    for (int e = 0; e < MAX_ELEM; ++e) {
        p.prog[e] = e < n_elem ? d_prog[e] : nullptr;
        p.variant[e] = e < n_elem ? variant[e] : -1;
        if (e < n_elem) use[variant[e]] = true;
    }
    cudaMemsetAsync(w.f_sorted, 0, sizeof(double) * 3 * (size_t)n, st);
    int launches = 0;
    if (use[ANG_BASE12]) launches += launch_one<SpecBase12>(p, st);
    if (use[ANG_WIDE32]) launches += launch_one<SpecWide32>(p, st);
    if (use[ANG_GENERIC]) launches += launch_one<SpecGeneric>(p, st);
    return launches;
}

}  // namespace nnp
