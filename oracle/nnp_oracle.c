/* nnp_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded FP64 CPU statement of what the hot path computes:
 * the Behler-Parrinello NNP energy and forces of PAPER.md section 3.1 / Fig. 1(b)
 * (L40: step 1 descriptors, step 2 atomic networks, step 3 forces), with the
 * formulas the paper leaves to its refs [18],[19] taken in the reading listed in
 * DESIGN.md "Readings" (= SURVEY.md 8(c) items 1-6, C1-C20).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call this file.  It shares no code, header,
 * table or constant with the CUDA library (paper_2002_00054_b200/csrc); the two
 * meet only in the tests, on arrays produced by workloads/.
 *
 * Everything is the definition written out: O(N) minimum-image scan per centre
 * (O(N^2) for all centres), one loop nest per symmetry function, the product
 * rule term by term for the gradients, no blocking, no caching of partial
 * results between symmetry functions, no reordering.
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): closed-form values for 2- and
 * 3-atom geometries (tests/golden/sf_closed_form.txt), minimum image through the
 * boundary, neighbour sets vs scipy's periodic k-d tree, MLP special cases and
 * finite differences in G, central finite differences of E vs analytic forces,
 * sum F = 0, translation / cube-rotation / free-rotation / permutation invariance,
 * and an independent PyTorch-autograd evaluation of the dense formula; the cell-prefiltered
 * neighbour search and oracle.forces_on (the glue of the full-size parity tests) against the
 * brute-force scan and the whole-system run (tests/test_oracle_cells_pins.py).
 * No function here is "parity unpinned".
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -shared -fPIC (see oracle/build.py).
 * -ffp-contract=off matters: the neighbour predicate must round every product and
 * sum individually (reading C7) so that neighbour SETS can be compared bit-exactly.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <time.h>

#define ORACLE_PI 3.14159265358979323846264338327950288

/* One symmetry function (own declaration; memory layout documented for ctypes).
 * kind 2: radial  G = sum_j exp(-eta (r_ij - rs)^2) fc(r_ij),   t_j = e1
 * kind 9: angular WIDE, as kind 3 without the r_jk terms (see sf_centre)
 * kind 3: angular G = 2^(1-zeta) sum_{j<k} (1 + lambda cos th)^zeta
 *                       exp(-eta (a^2+b^2+c^2)) fc(a) fc(b) fc(c),  {t_j,t_k} = {e1,e2}, c < rc
 * (n2p2 numbering, readings C2-C5). */
typedef struct {
    int32_t central, kind, e1, e2;
    double eta, rs, lambda, zeta;
} oracle_sf;

typedef struct {
    int32_t n_elem;
    double rc;
    int32_t n_sf;
    const oracle_sf* sf;          /* [n_sf]; order among equal `central` = order in G */
    const int32_t* n_layers;      /* [n_elem] number of weight layers (3 for in-25-25-1) */
    const int32_t* layer_sizes;   /* concatenated, n_layers[e]+1 entries per element     */
    const double* weights;        /* concatenated per element: W1[out][in], b1, W2, b2, ... */
    /* model generality (n2p2 scales / centres its symmetry functions and offers tanh):
     * network input x_s = sf_scale_s * (G_s - sf_shift_s); both concatenated per element in G order,
     * NULL = identity.  activation: 0 softplus (BASELINE.json), 1 tanh; output layer linear. */
    const double* sf_shift;
    const double* sf_scale;
    int32_t activation;
    /* per-SF cutoff radii (n2p2 gives every symmetry function its own rc): [n_sf] in the
     * order of `sf`, each 0 < sf_rc[q] <= rc; NULL = the one global rc.  The neighbourhood N(i) is still
     * the one of the global rc; an SF with a smaller rc simply has fc(r; sf_rc) = 0 beyond it. */
    const double* sf_rc;
} oracle_model;

static double now_s(void) {
    struct timespec ts;
    clock_gettime(CLOCK_MONOTONIC, &ts);
    return (double)ts.tv_sec + 1e-9 * (double)ts.tv_nsec;
}

/* ---- geometry (reading 1, C6, C7) ------------------------------------------- */

/* x <- x - L*floor(x/L), each operation individually rounded. */
void oracle_wrap(int64_t n, const double* pos, const double* box, double* out) {
    for (int64_t i = 0; i < n; ++i)
        for (int c = 0; c < 3; ++c) {
            double x = pos[3 * i + c], L = box[c];
            double q = floor(x / L);
            double p = L * q;
            out[3 * i + c] = x - p;
        }
}

/* d = x_j - x_i, then one conditional +-L per component (raw difference first). */
static void min_image(const double* xi, const double* xj, const double* box, double* d) {
    for (int c = 0; c < 3; ++c) {
        double L = box[c], h = 0.5 * L;
        double t = xj[c] - xi[c];
        if (t > h) t -= L;
        else if (t < -h) t += L;
        d[c] = t;
    }
}

static double norm2(const double* d) {
    double xx = d[0] * d[0], yy = d[1] * d[1], zz = d[2] * d[2];
    double s = xx + yy;
    return s + zz;                       /* (dx*dx + dy*dy) + dz*dz */
}

/* Row i of the neighbour list by brute force: all j != i with r^2 < rc^2 (strict),
 * ascending j.  `w` = wrapped positions.  Returns the count (may exceed cap; only
 * the first cap entries are written). */
int64_t oracle_neighbors_of(int64_t n, const double* w, const double* box, double rc,
                            int64_t i, int32_t* out, int64_t cap) {
    double rc2 = rc * rc, d[3];
    int64_t cnt = 0;
    for (int64_t j = 0; j < n; ++j) {
        if (j == i) continue;
        min_image(w + 3 * i, w + 3 * j, box, d);
        if (norm2(d) < rc2) {
            if (cnt < cap) out[cnt] = (int32_t)j;
            ++cnt;
        }
    }
    return cnt;
}

/* Full list, CSR.  offsets[n+1]; idx may be NULL (count only).  Returns total. */
int64_t oracle_neighbor_list(int64_t n, const double* pos, const double* box, double rc,
                             int64_t* offsets, int32_t* idx, int64_t cap) {
    double* w = (double*)malloc(sizeof(double) * 3 * (size_t)n);
    oracle_wrap(n, pos, box, w);
    int64_t total = 0;
    for (int64_t i = 0; i < n; ++i) {
        offsets[i] = total;
        int64_t room = (idx && total < cap) ? cap - total : 0;
        total += oracle_neighbors_of(n, w, box, rc, i, idx ? idx + total : NULL, room);
    }
    offsets[n] = total;
    free(w);
    return total;
}

/* ---- cell-prefiltered search (whole-system goldens only) ------------------------------
 * The SAME predicate (min_image + norm2 + strict <) applied to a candidate list instead of
 * to all N atoms: atoms are binned into nc = floor(L / (rc (1 + 1e-9))) >= 1 cells per
 * dimension (cell width >= rc (1 + 1e-9), so rounding in the bin index cannot matter) and
 * row i tests the atoms of the cells within +-1 of i's cell in every dimension, each
 * distinct periodic cell once.  Why this is a superset of N(i): |d| < rc implies
 * |d_c| < rc <= cell width in every component, and a component that took the +-L branch of
 * min_image has x_i, x_j within one cell width of opposite box faces -- in both cases the
 * cell indices differ by at most 1 modulo nc.  The candidates are then sorted ascending, so
 * the row equals oracle_neighbors_of() element by element.
 * It exists because the brute-force scan costs 25 ms per centre at 2.1 M atoms (15 core-hours
 * for the whole system); tests/golden/make_fullsize_golden.py uses it for whole-system sums
 * and re-checks rows against the brute-force scan while it runs.  Pinned bit-exact against
 * oracle_neighbors_of in tests/test_oracle_cells_pins.py (2-cell box, 1-cell dimensions,
 * 2x3x5 cells, atoms on box faces, every atom of configs[0] and of a 10-cell box). */
typedef struct {
    int64_t n;
    int32_t nc[3];
    int32_t* start;      /* [ncell + 1] */
    int32_t* items;      /* [n] atom indices, grouped by cell, ascending inside a cell */
    const double* w;     /* wrapped positions (not owned) */
    double box[3], rc;
} oracle_cells;

static int32_t cell_coord(double x, double L, int32_t nc) {
    int32_t c = (int32_t)floor(x / L * (double)nc);
    if (c < 0) c = 0;
    if (c > nc - 1) c = nc - 1;       /* x == L can come out of the wrap by rounding */
    return c;
}

oracle_cells* oracle_cells_build(int64_t n, const double* w, const double* box, double rc) {
    oracle_cells* C = (oracle_cells*)calloc(1, sizeof(oracle_cells));
    C->n = n; C->w = w; C->rc = rc;
    int64_t ncell = 1;
    for (int c = 0; c < 3; ++c) {
        C->box[c] = box[c];
        int32_t k = (int32_t)floor(box[c] / (rc * (1.0 + 1e-9)));
        if (k < 1) k = 1;
        if (k > 1024) k = 1024;
        C->nc[c] = k;
        ncell *= k;
    }
    C->start = (int32_t*)calloc((size_t)ncell + 1, sizeof(int32_t));
    C->items = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    int32_t* cid = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    for (int64_t i = 0; i < n; ++i) {
        int32_t cx = cell_coord(w[3 * i], box[0], C->nc[0]);
        int32_t cy = cell_coord(w[3 * i + 1], box[1], C->nc[1]);
        int32_t cz = cell_coord(w[3 * i + 2], box[2], C->nc[2]);
        cid[i] = (cz * C->nc[1] + cy) * C->nc[0] + cx;
        C->start[cid[i] + 1] += 1;
    }
    for (int64_t c = 0; c < ncell; ++c) C->start[c + 1] += C->start[c];
    int32_t* fill = (int32_t*)calloc((size_t)ncell, sizeof(int32_t));
    for (int64_t i = 0; i < n; ++i) C->items[C->start[cid[i]] + fill[cid[i]]++] = (int32_t)i;
    free(fill); free(cid);
    return C;
}

void oracle_cells_free(oracle_cells* C) {
    if (!C) return;
    free(C->start); free(C->items); free(C);
}

static int cmp_i32(const void* a, const void* b) {
    int32_t x = *(const int32_t*)a, y = *(const int32_t*)b;
    return (x > y) - (x < y);
}

/* the distinct cell coordinates within +-1 of c (periodic) along a dimension of nc cells */
static int stencil_1d(int32_t c, int32_t nc, int32_t* out) {
    if (nc <= 3) {                        /* 1, 2 or 3 cells: all of them, once */
        for (int32_t k = 0; k < nc; ++k) out[k] = k;
        return nc;
    }
    out[0] = (c + nc - 1) % nc; out[1] = c; out[2] = (c + 1) % nc;
    return 3;
}

/* Row i, same contract as oracle_neighbors_of (ascending j, count returned, first cap written). */
int64_t oracle_neighbors_of_cells(const oracle_cells* C, int64_t i, int32_t* out, int64_t cap) {
    const double* w = C->w;
    double rc2 = C->rc * C->rc, d[3];
    int32_t sx[3], sy[3], sz[3];
    int nx = stencil_1d(cell_coord(w[3 * i], C->box[0], C->nc[0]), C->nc[0], sx);
    int ny = stencil_1d(cell_coord(w[3 * i + 1], C->box[1], C->nc[1]), C->nc[1], sy);
    int nz = stencil_1d(cell_coord(w[3 * i + 2], C->box[2], C->nc[2]), C->nc[2], sz);
    int64_t cnt = 0, room = 64;
    int32_t* tmp = (int32_t*)malloc(sizeof(int32_t) * (size_t)room);
    for (int a = 0; a < nz; ++a)
        for (int b = 0; b < ny; ++b)
            for (int c = 0; c < nx; ++c) {
                int64_t cell = ((int64_t)sz[a] * C->nc[1] + sy[b]) * C->nc[0] + sx[c];
                for (int32_t q = C->start[cell]; q < C->start[cell + 1]; ++q) {
                    int64_t j = C->items[q];
                    if (j == i) continue;
                    min_image(w + 3 * i, w + 3 * j, C->box, d);
                    if (norm2(d) < rc2) {
                        if (cnt == room) { room *= 2; tmp = (int32_t*)realloc(tmp, sizeof(int32_t) * (size_t)room); }
                        tmp[cnt++] = (int32_t)j;
                    }
                }
            }
    qsort(tmp, (size_t)cnt, sizeof(int32_t), cmp_i32);
    for (int64_t k = 0; k < cnt && k < cap; ++k) out[k] = tmp[k];
    free(tmp);
    return cnt;
}

/* ---- cutoff (reading 2) ------------------------------------------------------- */

double oracle_fc(double r, double rc) {
    return r < rc ? 0.5 * (cos(ORACLE_PI * r / rc) + 1.0) : 0.0;
}

double oracle_dfc(double r, double rc) {
    return r < rc ? -0.5 * (ORACLE_PI / rc) * sin(ORACLE_PI * r / rc) : 0.0;
}

/* ---- symmetry functions of one centre (readings 3, 4) ---------------------------
 * u[m] = min-image vector centre -> neighbour m, tn[m] = its element.
 * G[s], s = position of the SF among those with central == tc.
 * If beta != NULL also accumulates forces: fi[3] on the centre, fn[m][3] on the
 * neighbours, F = - sum_s beta[s] * dG_s/dr   (reading 6). */
static void sf_centre(const oracle_model* M, int tc, int nn, const double* u, const int32_t* tn,
                      double* G, const double* beta, double* fi, double* fn) {
    int s = -1;
    for (int q = 0; q < M->n_sf; ++q) {
        const oracle_sf* f = &M->sf[q];
        if (f->central != tc) continue;
        ++s;
        const double rc = M->sf_rc ? M->sf_rc[q] : M->rc;     /* this SF's cutoff radius */
        double acc = 0.0;
        if (f->kind == 2) {
            for (int j = 0; j < nn; ++j) {
                if (tn[j] != f->e1) continue;
                const double* uj = u + 3 * j;
                double r = sqrt(uj[0] * uj[0] + uj[1] * uj[1] + uj[2] * uj[2]);
                double dr = r - f->rs;
                double ex = exp(-f->eta * dr * dr);
                double c = oracle_fc(r, rc);
                acc += ex * c;
                if (beta) {
                    /* d/dr [ex * fc] = ex * (fc' - 2 eta (r - rs) fc);  dr/dr_j = u/r */
                    double dg = ex * (oracle_dfc(r, rc) - 2.0 * f->eta * dr * c);
                    for (int x = 0; x < 3; ++x) {
                        double gx = dg * uj[x] / r;       /* dG/dr_j ;  dG/dr_i = -gx */
                        fn[3 * j + x] -= beta[s] * gx;
                        fi[x] += beta[s] * gx;
                    }
                }
            }
        } else { /* kind 3 (angular narrow) or kind 9 (angular WIDE, n2p2 numbering):
                  *   G = 2^(1-zeta) sum_{j<k} (1 + lambda cos)^zeta exp(-eta (a^2 + b^2)) fc(a) fc(b)
                  * -- no r_jk term and no r_jk cutoff: every pair of neighbours of the two elements counts */
            const int wide = (f->kind == 9);
            double pref = pow(2.0, 1.0 - f->zeta);
            for (int j = 0; j < nn; ++j)
                for (int k = j + 1; k < nn; ++k) {
                    int tj = tn[j], tk = tn[k];
                    if (!((tj == f->e1 && tk == f->e2) || (tj == f->e2 && tk == f->e1))) continue;
                    const double* uu = u + 3 * j;
                    const double* vv = u + 3 * k;
                    double ww[3] = {vv[0] - uu[0], vv[1] - uu[1], vv[2] - uu[2]};
                    double a2 = uu[0] * uu[0] + uu[1] * uu[1] + uu[2] * uu[2];
                    double b2 = vv[0] * vv[0] + vv[1] * vv[1] + vv[2] * vv[2];
                    double c2 = ww[0] * ww[0] + ww[1] * ww[1] + ww[2] * ww[2];
                    double a = sqrt(a2), b = sqrt(b2), c = sqrt(c2);
                    if (!wide && !(c < rc)) continue;             /* narrow: needs r_jk < rc */
                    double ct = (uu[0] * vv[0] + uu[1] * vv[1] + uu[2] * vv[2]) / (a * b);
                    double base = 1.0 + f->lambda * ct;
                    double P = pref * pow(base, f->zeta);
                    double X = exp(-f->eta * (wide ? a2 + b2 : a2 + b2 + c2));
                    double fa = oracle_fc(a, rc), fb = oracle_fc(b, rc), fcc = wide ? 1.0 : oracle_fc(c, rc);
                    double C = fa * fb * fcc;
                    acc += P * X * C;
                    if (beta) {
                        double dP = pref * f->zeta * f->lambda * pow(base, f->zeta - 1.0); /* dP/dcos */
                        double dfa = oracle_dfc(a, rc), dfb = oracle_dfc(b, rc), dfc = wide ? 0.0 : oracle_dfc(c, rc);
                        const double wq = wide ? 0.0 : 1.0;       /* weight of the c^2 term in the exponent */
                        for (int x = 0; x < 3; ++x) {
                            /* cos = u.v/(ab) */
                            double dct_du = vv[x] / (a * b) - ct * uu[x] / a2;
                            double dct_dv = uu[x] / (a * b) - ct * vv[x] / b2;
                            /* X = exp(-eta(a2+b2+c2)), c2 = |v-u|^2 */
                            double dX_du = X * (-f->eta) * (2.0 * uu[x] - wq * 2.0 * ww[x]);
                            double dX_dv = X * (-f->eta) * (2.0 * vv[x] + wq * 2.0 * ww[x]);
                            /* C = fc(a) fc(b) fc(c) */
                            double dC_du = dfa * (uu[x] / a) * fb * fcc + fa * fb * dfc * (-ww[x] / c);
                            double dC_dv = fa * dfb * (vv[x] / b) * fcc + fa * fb * dfc * (ww[x] / c);
                            double dg_du = dP * dct_du * X * C + P * dX_du * C + P * X * dC_du;
                            double dg_dv = dP * dct_dv * X * C + P * dX_dv * C + P * X * dC_dv;
                            /* r_j = r_i + u, r_k = r_i + v */
                            fn[3 * j + x] -= beta[s] * dg_du;
                            fn[3 * k + x] -= beta[s] * dg_dv;
                            fi[x] += beta[s] * (dg_du + dg_dv);
                        }
                    }
                }
        }
        if (G) G[s] = acc;
    }
}

/* ---- atomic network (reading 5) -------------------------------------------------
 * softplus hidden layers, linear output; returns E and dE/dG (beta).             */
static double softplus(double x) { return fmax(x, 0.0) + log1p(exp(-fabs(x))); }
static double sigmoid(double x) { return 1.0 / (1.0 + exp(-x)); }

static double act_f(int kind, double z) { return kind == 1 ? tanh(z) : softplus(z); }
static double act_d(int kind, double z) {
    if (kind == 1) { const double t = tanh(z); return 1.0 - t * t; }
    return sigmoid(z);
}

/* E = NN(x), x_s = scale_s (G_s - shift_s);  beta_s = dE/dG_s = scale_s dE/dx_s */
void oracle_mlp2(int32_t n_layers, const int32_t* sizes, const double* wts, const double* G,
                 const double* shift /* may be NULL */, const double* scale /* may be NULL */, int32_t activation,
                 double* e_out, double* beta /* may be NULL */) {
    int maxw = 0;
    for (int l = 0; l <= n_layers; ++l)
        if (sizes[l] > maxw) maxw = sizes[l];
    double* act = (double*)calloc((size_t)(n_layers + 1) * maxw, sizeof(double)); /* activations */
    double* pre = (double*)calloc((size_t)(n_layers + 1) * maxw, sizeof(double)); /* pre-activations */
    for (int i = 0; i < sizes[0]; ++i) act[i] = (scale ? scale[i] : 1.0) * (G[i] - (shift ? shift[i] : 0.0));
    const double* p = wts;
    for (int l = 0; l < n_layers; ++l) {
        int nin = sizes[l], nout = sizes[l + 1];
        const double* W = p;
        const double* b = p + (size_t)nout * nin;
        p = b + nout;
        for (int o = 0; o < nout; ++o) {
            double z = b[o];
            for (int i = 0; i < nin; ++i) z += W[(size_t)o * nin + i] * act[(size_t)l * maxw + i];
            pre[(size_t)(l + 1) * maxw + o] = z;
            act[(size_t)(l + 1) * maxw + o] = (l == n_layers - 1) ? z : act_f(activation, z);
        }
    }
    *e_out = act[(size_t)n_layers * maxw + 0];
    if (beta) {
        /* back-propagate d E / d act_l */
        double* g = (double*)calloc((size_t)maxw, sizeof(double));
        double* gp = (double*)calloc((size_t)maxw, sizeof(double));
        g[0] = 1.0;
        /* recompute layer pointers from the back */
        const double** Wl = (const double**)malloc(sizeof(double*) * n_layers);
        p = wts;
        for (int l = 0; l < n_layers; ++l) {
            Wl[l] = p;
            p += (size_t)sizes[l + 1] * sizes[l] + sizes[l + 1];
        }
        for (int l = n_layers - 1; l >= 0; --l) {
            int nin = sizes[l], nout = sizes[l + 1];
            for (int i = 0; i < nin; ++i) gp[i] = 0.0;
            for (int o = 0; o < nout; ++o) {
                double dz = g[o] * ((l == n_layers - 1) ? 1.0 : act_d(activation, pre[(size_t)(l + 1) * maxw + o]));
                for (int i = 0; i < nin; ++i) gp[i] += Wl[l][(size_t)o * nin + i] * dz;
            }
            for (int i = 0; i < nin; ++i) g[i] = gp[i];
        }
        for (int i = 0; i < sizes[0]; ++i) beta[i] = (scale ? scale[i] : 1.0) * g[i];
        free(g); free(gp); free(Wl);
    }
    free(act); free(pre);
}

/* the BASELINE.json network: softplus, unscaled input */
void oracle_mlp(int32_t n_layers, const int32_t* sizes, const double* wts, const double* G,
                double* e_out, double* beta /* may be NULL */) {
    oracle_mlp2(n_layers, sizes, wts, G, NULL, NULL, 0, e_out, beta);
}

static void element_net(const oracle_model* M, int e, int32_t* n_layers, const int32_t** sizes,
                        const double** wts) {
    const int32_t* ls = M->layer_sizes;
    const double* w = M->weights;
    for (int q = 0; q < e; ++q) {
        int nl = M->n_layers[q];
        for (int l = 0; l < nl; ++l) w += (size_t)ls[l + 1] * ls[l] + ls[l + 1];
        ls += nl + 1;
    }
    *n_layers = M->n_layers[e];
    *sizes = ls;
    *wts = w;
}

int32_t oracle_n_sf_of(const oracle_model* M, int e) {
    int n = 0;
    for (int q = 0; q < M->n_sf; ++q) n += (M->sf[q].central == e);
    return n;
}

/* ---- the path for a set of centres ------------------------------------------------
 * For every selected centre i (sel == NULL: all atoms, n_sel = n):
 *   N(i) by brute force, G_i, E_i = NN_{t_i}(G_i), beta_i = dE_i/dG_i, and - if F is
 *   given - the forces  -beta_i . dG_i/dr  added to F[i] and F[j in N(i)].
 * With all atoms selected F is the total force and sum(e_atom) the total energy.
 * Outputs (any may be NULL): e_atom[n_sel], G[n_sel][g_stride], dEdG[n_sel][g_stride],
 * nbr_count[n_sel], F[n][3] (accumulated into - caller zeroes), timing[2] =
 * {seconds in neighbour search, seconds in SF + NN + forces}.
 * search / row_off / row_idx: see the parameter comments (row_idx holds at most row_cap entries; row_off is
 * always complete, so a second call with a big enough buffer gets every row).
 * Returns 0, or -1 if a type is out of range / box < 2 rc. */
int32_t oracle_centres_ex(const oracle_model* M, int64_t n, const double* pos, const int32_t* type,
                          const double* box, int64_t n_sel, const int64_t* sel,
                          double* e_atom, double* G, double* dEdG, int64_t g_stride,
                          int32_t* nbr_count, double* F, double* timing,
                          int32_t search /* 0 brute-force scan (the definition), 1 cell-prefiltered (same rows) */,
                          int64_t* row_off /* [n_sel + 1] or NULL */, int32_t* row_idx /* or NULL */, int64_t row_cap) {
    for (int c = 0; c < 3; ++c)
        if (!(box[c] >= 2.0 * M->rc)) return -1;
    for (int64_t i = 0; i < n; ++i)
        if (type[i] < 0 || type[i] >= M->n_elem) return -1;
    double* w = (double*)malloc(sizeof(double) * 3 * (size_t)n);
    oracle_wrap(n, pos, box, w);
    int32_t* nb = (int32_t*)malloc(sizeof(int32_t) * (size_t)n);
    oracle_cells* cells = search == 1 ? oracle_cells_build(n, w, box, M->rc) : NULL;
    int64_t row_total = 0;
    double t_nbr = 0.0, t_rest = 0.0;
    int maxsf = 0;
    for (int e = 0; e < M->n_elem; ++e) {
        int k = oracle_n_sf_of(M, e);
        if (k > maxsf) maxsf = k;
    }
    double* Gi = (double*)malloc(sizeof(double) * (size_t)(maxsf + 1));
    double* bi = (double*)malloc(sizeof(double) * (size_t)(maxsf + 1));
    for (int64_t q = 0; q < n_sel; ++q) {
        int64_t i = sel ? sel[q] : q;
        double t0 = now_s();
        int64_t nn = cells ? oracle_neighbors_of_cells(cells, i, nb, n) : oracle_neighbors_of(n, w, box, M->rc, i, nb, n);
        if (row_off) {                        /* the neighbour rows of the selected centres, CSR */
            row_off[q] = row_total;
            for (int64_t m = 0; m < nn; ++m)
                if (row_idx && row_total + m < row_cap) row_idx[row_total + m] = nb[m];
            row_total += nn;
        }
        double* u = (double*)malloc(sizeof(double) * 3 * (size_t)(nn + 1));
        int32_t* tn = (int32_t*)malloc(sizeof(int32_t) * (size_t)(nn + 1));
        for (int64_t m = 0; m < nn; ++m) {
            min_image(w + 3 * i, w + 3 * (int64_t)nb[m], box, u + 3 * m);
            tn[m] = type[nb[m]];
        }
        double t1 = now_s();
        int tc = type[i];
        int nsf = oracle_n_sf_of(M, tc);
        sf_centre(M, tc, (int)nn, u, tn, Gi, NULL, NULL, NULL);
        int32_t nl; const int32_t* sizes; const double* wts;
        element_net(M, tc, &nl, &sizes, &wts);
        double e;
        int sf_off = 0;                       /* this element's slice of sf_shift / sf_scale */
        for (int q2 = 0; q2 < tc; ++q2) sf_off += oracle_n_sf_of(M, q2);
        oracle_mlp2(nl, sizes, wts, Gi, M->sf_shift ? M->sf_shift + sf_off : NULL,
                    M->sf_scale ? M->sf_scale + sf_off : NULL, M->activation, &e, bi);
        if (e_atom) e_atom[q] = e;
        if (G) for (int s = 0; s < nsf; ++s) G[q * g_stride + s] = Gi[s];
        if (dEdG) for (int s = 0; s < nsf; ++s) dEdG[q * g_stride + s] = bi[s];
        if (nbr_count) nbr_count[q] = (int32_t)nn;
        if (F) {
            double fi[3] = {0.0, 0.0, 0.0};
            double* fn = (double*)calloc(3 * (size_t)(nn + 1), sizeof(double));
            sf_centre(M, tc, (int)nn, u, tn, NULL, bi, fi, fn);
            for (int x = 0; x < 3; ++x) F[3 * i + x] += fi[x];
            for (int64_t m = 0; m < nn; ++m)
                for (int x = 0; x < 3; ++x) F[3 * (int64_t)nb[m] + x] += fn[3 * m + x];
            free(fn);
        }
        free(u); free(tn);
        double t2 = now_s();
        t_nbr += t1 - t0;
        t_rest += t2 - t1;
    }
    if (row_off) row_off[n_sel] = row_total;
    if (timing) { timing[0] = t_nbr; timing[1] = t_rest; }
    oracle_cells_free(cells);
    free(Gi); free(bi); free(nb); free(w);
    return 0;
}

/* the definition: brute-force neighbour scan, no row export */
int32_t oracle_centres(const oracle_model* M, int64_t n, const double* pos, const int32_t* type,
                       const double* box, int64_t n_sel, const int64_t* sel,
                       double* e_atom, double* G, double* dEdG, int64_t g_stride,
                       int32_t* nbr_count, double* F, double* timing) {
    return oracle_centres_ex(M, n, pos, type, box, n_sel, sel, e_atom, G, dEdG, g_stride, nbr_count, F, timing,
                             0, NULL, NULL, 0);
}
