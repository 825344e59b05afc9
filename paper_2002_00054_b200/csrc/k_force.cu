// k_force.cu -- S4: forces  F_m = - sum_i sum_s beta_is dG_is/dr_m  with beta = dE_i/dG_i from the
// network kernel and dG/dr RECOMPUTED here, never stored (PAPER.md L40 step 3, L56-58 "store and
// move as little data as possible, recomputing where necessary", L98, L124).  This holds "the
// dominant angular force loop" (L116) and is the hottest kernel of the path.
//
// GENERIC path: any symmetry-function table.  Tables with the structure of a compile-time Spec
// (angular.cuh) run on the lane-owned fast path, k_force2.cu.
// One warp per centre i, same staging / round enumeration / compaction as k_sf.cu.  For a
// triplet (i; j,k) with u = r_j - r_i, v = r_k - r_i, w = v - u the beta-weighted gradient is
//     dg/du = f_uu u + f_uv v - f_w w,      dg/dv = f_vv v + f_uv u + f_w w
// (DESIGN.md "Force algebra"), so  F_j = -s1 u + s3 v,  F_k = -s2 v + s3 u  with
// s1 = f_uu + f_w, s2 = f_vv + f_w, s3 = f_w - f_uv.  Per neighbour SLOT the kernel accumulates
// the scalar A = sum s1 and the vector V = sum s3 (partner vector) in shared memory and forms
// F_slot = V - A u once per centre; the slot forces are flushed with one global FP64 RED per
// component per neighbour.  Slot accumulation is a plain read-modify-write done one COLOUR at
// a time (angular.cuh): pairs of equal colour never share a slot, and a warp owns its slots, so
// no shared-memory atomics are needed (the first version's FP64 shared atomicAdd = CAS loops
// took >35 % of the stall samples and ran 2.8 iterations on average; profiles/r1_*).
#include "angular.cuh"
#include "geometry.cuh"

namespace nnp {

constexpr int FC_WARPS = 4;
constexpr double PI_D = 3.14159265358979323846;

struct ForceParams {
    int64_t n;
    int n_elem, ncell, stride, cap, g_stride;
    double rc, rc2, inv_rc, k2;          // k2 = (pi / (2 rc))^2
    double box[3], half[3];
    const double *sx, *sy, *sz;
    const int32_t *cell_start, *nbr, *nbr_cnt;
    const double* dEdG;
    double* f_sorted;
    int fixed;                           // 1: fixed-point force accumulation (nnp_internal.h force_add)
    int32_t *status, *sticky;
    const ElemProgram* prog[MAX_ELEM];
    int variant[MAX_ELEM];
    int radial_only[MAX_ELEM];           // 1: run only the radial block for this element (per-SF radial radii of a lane-owned element)
};

// per-warp shared-memory footprint (bytes): six double2 planes (geometry, cutoff, Gaussian, two
// accumulators), the FP32 screening copy, the coefficient tables of all pair groups, and the beta row
// which later doubles as the 64-entry pair queue
template <class Spec>
__host__ __device__ constexpr int bt_stride() { return Spec::NACC + 1; }   // +1: groups land on different banks

template <class Spec>
__host__ __device__ constexpr size_t force_warp_smem(int cap, int g_stride, int n_elem) {
    const size_t capa = (size_t)((cap + 3) & ~3);
    const size_t npair = (size_t)n_elem * (n_elem + 1) / 2;
    size_t b = capa * (6 * 16 + 12);
    b += npair * bt_stride<Spec>() * 16;
    const size_t rowq = (size_t)g_stride * 8 > 256 ? (size_t)g_stride * 8 : 256;
    b += rowq;
    return (b + 15) / 16 * 16;
}

// shared per-slot accumulators: F_slot = V - A * u
struct SlotAcc {
    double2* av;   // (A, Vx)
    double2* yz;   // (Vy, Vz)
};

// One triplet's  F_j = -s1 u + s3 v  and  F_k = -s2 v + s3 u  into the shared slot accumulators (A, V).
__device__ __forceinline__ void slot_updates(const double2 j0, const double2 j1, const double2 k0, const double2 k1, double s1,
                                             double s2, double s3, const SlotAcc& acc, int j, int k, int col, bool active) {
    // colour passes: entries of one colour have pairwise distinct j and pairwise distinct k
    unsigned pend = __ballot_sync(0xffffffffu, active);
    while (pend) {
        const int c = __shfl_sync(0xffffffffu, col, __ffs(pend) - 1);
        const bool mine = active && col == c;
        if (mine) {
            double2 a = acc.av[j], b = acc.yz[j];
            a.x += s1;
            a.y = fma(s3, k0.x, a.y);
            b.x = fma(s3, k0.y, b.x);
            b.y = fma(s3, k1.x, b.y);
            acc.av[j] = a;
            acc.yz[j] = b;
        }
        __syncwarp();
        if (mine) {
            double2 a = acc.av[k], b = acc.yz[k];
            a.x += s2;
            a.y = fma(s3, j0.x, a.y);
            b.x = fma(s3, j0.y, b.x);
            b.y = fma(s3, j1.x, b.y);
            acc.av[k] = a;
            acc.yz[k] = b;
        }
        __syncwarp();
        pend &= ~__ballot_sync(0xffffffffu, mine);
    }
}

// From Z0 = sum beta P Y, Z1 = sum beta P' Y, Z2 = sum eta beta P Y  (Y = product of the three
// bare Gaussians) to the slot updates.  fcc = fc(c), dfc = fc'(c)/c.
__device__ __forceinline__ void triplet_forces(const double2 j0, const double2 j1, const double2 j2, const double2 k0,
                                               const double2 k1, const double2 k2, double fcc, double dfc, double cosv,
                                               double iab, double Z0, double Z1, double Z2, double W0, double W1,
                                               double W2, const SlotAcc& acc, int j, int k, int col, bool active) {
    const double fa = j2.x, dfa = j2.y, fb = k2.x, dfb = k2.y, ia = j1.y, ib = k1.y;
    const double fab = fa * fb;
    const double C = fab * fcc;
    const double t2 = (C + C) * Z2;
    const double f_w = fma(fab * dfc, Z0, -t2);
    const double q = Z1 * C;
    const double qc = q * cosv;
    const double f_uu = fma(-qc, ia * ia, fma((dfa * fb) * fcc, Z0, -t2));
    const double f_vv = fma(-qc, ib * ib, fma((fa * dfb) * fcc, Z0, -t2));
    // wide SFs (kind 9): the same sums W0, W1, W2 over their own list, without any r_jk dependence
    const double tw = (fab + fab) * W2;
    const double qw = W1 * fab;
    const double qwc = qw * cosv;
    const double g_uu = fma(-qwc, ia * ia, fma(dfa * fb, W0, -tw));
    const double g_vv = fma(-qwc, ib * ib, fma(fa * dfb, W0, -tw));
    const double s1 = f_uu + f_w + g_uu, s2 = f_vv + f_w + g_vv, s3 = fma(-(q + qw), iab, f_w);
    slot_updates(j0, j1, k0, k1, s1, s2, s3, acc, j, k, col, active);
}

struct ForceTripletGeneric {
    const Nbh& nb;
    SlotAcc acc;
    const AngularSF* list;
    int nsf;
    const double* brow;   // beta row of the centre (shared memory)
    double k2, rc2;
    bool own;             // the SFs carry their own cutoff radii (ElemProgram::per_sf_rc)

    __device__ __forceinline__ void operator()(int j, int k, int col, bool active) {
        const double2 j0 = nb.p0[j], j1 = nb.p1[j], j2 = nb.p2[j];
        const double2 k0 = nb.p0[k], k1 = nb.p1[k], kk2 = nb.p2[k];
        const double wx = k0.x - j0.x, wy = k0.y - j0.y, wz = k1.x - j1.x;
        const double c2 = fma(wx, wx, fma(wy, wy, wz * wz));
        double Cc, Sc;
        cos_sinc(c2 * k2, Cc, Sc);
        double fcc = Cc * Cc;
        double dfc = (-2.0 * k2) * (Cc * Sc);
        if (!active || !(c2 < rc2)) { fcc = 0.0; dfc = 0.0; }
        const double iab = j1.y * k1.y;
        const double cosv = fma(j0.x, k0.x, fma(j0.y, k0.y, j1.x * k1.x)) * iab;
        const double a2 = 1.0 / (j1.y * j1.y), b2 = 1.0 / (k1.y * k1.y);
        const double r2ab = a2 + b2;
        const double r2sum = r2ab + c2;
        if (own) {
            // every SF has its own fc(.; rc_s): no common cutoff factor to pull out, the three slot scalars are summed SF by SF
            const double a2j = fma(j0.x, j0.x, fma(j0.y, j0.y, j1.x * j1.x)), a2k = fma(k0.x, k0.x, fma(k0.y, k0.y, k1.x * k1.x));
            const double ia2 = j1.y * j1.y, ib2 = k1.y * k1.y;
            double s1 = 0.0, s2 = 0.0, s3 = 0.0, en = -1.0, ew = -1.0, Yn = 0.0, Yw = 0.0;
            for (int s = 0; s < nsf; ++s) {
                const AngularSF f = list[s];
                const double base = 1.0 + (double)f.lam * cosv;
                double pd = 1.0, bb = base;
                for (int z = f.izeta - 1; z > 0; z >>= 1) {
                    if (z & 1) pd *= bb;
                    bb *= bb;
                }
                double fa, dfa, fb, dfb, fcs = 1.0, dfcs = 0.0;
                fc_dfc_own(a2j, f.rc2, f.k2, fa, dfa);
                fc_dfc_own(a2k, f.rc2, f.k2, fb, dfb);
                if (!f.wide) fc_dfc_own(c2, f.rc2, f.k2, fcs, dfcs);
                double Y;
                if (f.wide) {
                    if (f.eta != ew) { ew = f.eta; Yw = exp_small(fmax(-f.eta * (a2j + a2k), -700.0)); }
                    Y = Yw;
                } else {
                    if (f.eta != en) { en = f.eta; Yn = exp_small(fmax(-f.eta * (a2j + a2k + c2), -700.0)); }
                    Y = Yn;
                }
                const double bc = brow[f.g] * f.coef;
                const double t0 = bc * (pd * base) * Y, t1 = bc * (double)(f.izeta * f.lam) * pd * Y;
                const double fab = fa * fb, C = fab * fcs;
                const double t2 = (C + C) * (f.eta * t0);
                const double fw = f.wide ? 0.0 : fma(fab * dfcs, t0, -t2);
                const double q = t1 * C, qc = q * cosv;
                s1 += fma(-qc, ia2, fma((dfa * fb) * fcs, t0, -t2)) + fw;
                s2 += fma(-qc, ib2, fma((fa * dfb) * fcs, t0, -t2)) + fw;
                s3 += fma(-q, iab, fw);
            }
            slot_updates(j0, j1, k0, k1, s1, s2, s3, acc, j, k, col, active);
            return;
        }
        double Z0 = 0.0, Z1 = 0.0, Z2 = 0.0, W0 = 0.0, W1 = 0.0, W2 = 0.0;
        double en = -1.0, ew = -1.0, Yn = 0.0, Yw = 0.0;
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
            double Y;           // exp(-eta r^2), shared by consecutive SFs of equal eta
            if (f.wide) {
                if (f.eta != ew) { ew = f.eta; Yw = exp_small(fmax(-f.eta * r2ab, -700.0)); }
                Y = Yw;
            } else {
                if (f.eta != en) { en = f.eta; Yn = exp_small(fmax(-f.eta * r2sum, -700.0)); }
                Y = Yn;
            }
            const double bc = brow[f.g] * f.coef;
            const double t0 = bc * pwv * Y, t1 = bc * (double)(f.izeta * f.lam) * pd * Y;
            if (f.wide) {
                W0 += t0;
                W1 += t1;
                W2 = fma(f.eta, t0, W2);
            } else {
                Z0 += t0;
                Z1 += t1;
                Z2 = fma(f.eta, t0, Z2);
            }
        }
        triplet_forces(j0, j1, j2, k0, k1, kk2, fcc, dfc, cosv, iab, Z0, Z1, Z2, W0, W1, W2, acc, j, k, col, active);
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
    if (p.variant[tc] != Spec::ID && p.radial_only[tc] == 0) return;
    const ElemProgram* __restrict__ prog = p.prog[tc];
    const bool radial_only = p.radial_only[tc] != 0;      // see k_sf.cu: the radial forces of a lane-owned element with own radial radii

    const int capa = (p.cap + 3) & ~3;
    const int npair = p.n_elem * (p.n_elem + 1) / 2;
    unsigned char* base = smem_raw + (size_t)wid * force_warp_smem<Spec>(p.cap, p.g_stride, p.n_elem);
    Nbh nb;
    nb.p0 = reinterpret_cast<double2*>(base);
    nb.p1 = nb.p0 + capa;
    nb.p2 = nb.p1 + capa;
    nb.p3 = nb.p2 + capa;
    SlotAcc acc;
    acc.av = nb.p3 + capa;
    acc.yz = acc.av + capa;
    double2* bt = acc.yz + capa;
    nb.fxy = reinterpret_cast<float2*>(bt + npair * bt_stride<Spec>());
    nb.fz = reinterpret_cast<float*>(nb.fxy + capa);
    double* brow = reinterpret_cast<double*>(nb.fz + capa);
    PairQueue Q;
    Q.q = reinterpret_cast<uint32_t*>(brow);   // the beta row is dead once the tables are built
    Q.head = 0;
    Q.n = 0;

    int seg[MAX_ELEM + 1];
    seg[0] = 0;
#pragma unroll
    for (int e = 0; e < MAX_ELEM; ++e) seg[e + 1] = seg[e] + p.nbr_cnt[(size_t)i * MAX_ELEM + e];
    const int ntot = seg[MAX_ELEM];

    for (int s = lane; s < p.g_stride; s += 32) brow[s] = p.dEdG[(size_t)i * p.g_stride + s];
    __syncwarp();

    // ---- stage the neighbourhood; the radial force  F_j = -R u  seeds the scalar accumulator A ---
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
            const double a2 = fma(dx, dx, fma(dy, dy, dz * dz));
            const double ia = rsqrt(a2);
            const double a = a2 * ia;
            double Ca, Sa;
            cos_sinc(a2 * p.k2, Ca, Sa);
            const double fa = Ca * Ca;                          // fc(a)
            const double dfa_a = (-2.0 * p.k2) * (Ca * Sa);     // fc'(a)/a
            nb.p0[m] = make_double2(dx, dy);
            nb.p1[m] = make_double2(dz, ia);
            nb.p2[m] = make_double2(fa, dfa_a);
            nb.fxy[m] = make_float2((float)dx, (float)dy);
            nb.fz[m] = (float)dz;
            if constexpr (Spec::NETA > 0) nb.p3[m] = make_double2(exp_small(-eta0 * a2), 0.0);
            // R = sum_r beta_r exp(-eta d^2) (fc'(a) - 2 eta d fc(a)) / a,  d = a - rs
            double R = 0.0;
            for (int r = 0; r < nr; ++r) {
                const RadialSF f = prog->rad[off + r];
                const double d = a - f.rs;
                const double ex = exp_small(fmax(-f.eta * d * d, -700.0));
                double fs = fa, dfs = dfa_a;
                if (prog->per_sf_rc) fc_dfc_own(a2, f.rc2, f.k2, fs, dfs);
                R = fma(brow[f.g] * ex, fma(-2.0 * f.eta * d, fs * ia, dfs), R);
            }
            acc.av[m] = make_double2(R, 0.0);
            acc.yz[m] = make_double2(0.0, 0.0);
        }
    }
    __syncwarp();

    // ---- angular part ---------------------------------------------------------------------------
    const float rc2f = screen_rc2(p.rc2);
    if (!radial_only) {
        // generic tables: per pair group, walking the SF list; the beta row stays live, so the queue
        // sits in the (unused) p3 plane
        Q.q = reinterpret_cast<uint32_t*>(nb.p3);
        for (int e1 = 0; e1 < p.n_elem; ++e1)
            for (int e2 = e1; e2 < p.n_elem; ++e2) {
                const int pr = pair_index(e1, e2, p.n_elem);
                const int na = prog->n_ang[pr];
                if (na == 0) continue;
                ForceTripletGeneric f{nb, acc, prog->ang + prog->ang_off[pr], na, brow, p.k2, p.rc2, prog->per_sf_rc != 0};
                const float rs = group_has_wide(prog->ang + prog->ang_off[pr], na) ? 3.0e38f : rc2f;   // wide SFs: no r_jk screen
                if (e1 == e2) pairs_within(nb, seg[e1], seg[e1 + 1] - seg[e1], rs, Q, lane, f);
                else pairs_between(nb, seg[e1], seg[e1 + 1] - seg[e1], seg[e2], seg[e2 + 1] - seg[e2], rs, Q, lane, f);
            }
    }
    __syncwarp();

    // ---- flush: F_slot = V - A u; one global FP64 RED per component; the centre gets minus the sum
    double fx = 0.0, fy = 0.0, fz = 0.0;
    for (int m = lane; m < ntot; m += 32) {
        const int j = row[m];
        const double2 u0 = nb.p0[m], av = acc.av[m], yz = acc.yz[m];
        const double uz = nb.p1[m].x;
        const double ax = fma(-av.x, u0.x, av.y), ay = fma(-av.x, u0.y, yz.x), az = fma(-av.x, uz, yz.y);
        force_add(p, 3 * (size_t)j + 0, ax);
        force_add(p, 3 * (size_t)j + 1, ay);
        force_add(p, 3 * (size_t)j + 2, az);
        fx -= ax; fy -= ay; fz -= az;
    }
    fx = warp_sum(fx); fy = warp_sum(fy); fz = warp_sum(fz);
    if (lane == 0) {
        force_add(p, 3 * (size_t)i + 0, fx);
        force_add(p, 3 * (size_t)i + 1, fy);
        force_add(p, 3 * (size_t)i + 2, fz);
    }
}

template <class Spec>
static int launch_one(const ForceParams& p, cudaStream_t st) {
    const size_t smem = FC_WARPS * force_warp_smem<Spec>(p.cap, p.g_stride, p.n_elem);
    static unsigned long long configured = 0ull;      // per device (opt_in_smem)
    opt_in_smem(k_force<Spec>, &configured);
    const unsigned nb = (unsigned)((p.n + FC_WARPS - 1) / FC_WARPS);
    k_force<Spec><<<nb, FC_WARPS * 32, smem, st>>>(p);
    return 1;
}

int launch_force(const Workspace& w, const Grid& g, int64_t n, int n_elem, const ElemProgram* const* d_prog,
                 const int* variant, const PassInfo& passes, double rc, int stride, int max_nbr, int g_stride, int precision,
                 cudaStream_t st) {
    if (n == 0) return 0;
    ForceParams p;
    p.n = n; p.n_elem = n_elem; p.ncell = g.ncell; p.stride = stride; p.cap = max_nbr; p.g_stride = g_stride;
    p.rc = rc; p.rc2 = rc * rc; p.inv_rc = 1.0 / rc; p.k2 = (PI_D / (2.0 * rc)) * (PI_D / (2.0 * rc));
    for (int c = 0; c < 3; ++c) { p.box[c] = g.box[c]; p.half[c] = g.half[c]; }
    p.sx = w.sx; p.sy = w.sy; p.sz = w.sz;
    p.cell_start = w.cell_start; p.nbr = w.nbr; p.nbr_cnt = w.nbr_cnt; p.dEdG = w.dEdG; p.f_sorted = w.f_sorted;
    p.fixed = passes.fixed_forces; p.status = w.status; p.sticky = w.sticky;
    bool use[ANG_NVARIANT] = {};
    for (int e = 0; e < MAX_ELEM; ++e) {
        p.prog[e] = e < n_elem ? d_prog[e] : nullptr;
        p.variant[e] = e < n_elem ? (variant[e] & 255) : -1;      // bit 8 = tiny_exp flag (fast launchers)
        p.radial_only[e] = (e < n_elem && (variant[e] & 255) != ANG_GENERIC && passes.radial_own[e]) ? 1 : 0;
        if (e < n_elem) use[variant[e] & 255] = true;
        if (p.radial_only[e]) use[ANG_GENERIC] = true;
    }
    cudaMemsetAsync(w.f_sorted, 0, sizeof(double) * 3 * (size_t)n, st);
    int launches = 0;
    if (use[ANG_BASE12] || use[ANG_WIDE32] || use[ANG_FREE32] || use[ANG_FREE16] || use[ANG_MULTI])     // specialised tables: lane-owned design (k_force2.cu)
        launches += launch_force2(w, g, n, n_elem, d_prog, variant, passes, rc, stride, max_nbr, g_stride, precision, st);
    if (use[ANG_GENERIC]) launches += launch_one<SpecGeneric>(p, st);
    return launches;
}

}  // namespace nnp
