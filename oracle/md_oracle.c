/*
 * md_oracle.c -- fp64 CPU ORACLE for the short-range force path of arXiv 1401.4350.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load this file.  It shares no code, header,
 * table or helper with the CUDA path under paper_1401_4350_b200/ and neither imports
 * the other.  It is plain, slow and written to be checked against the paper by eye;
 * it is never tuned.
 *
 * What it computes (citations: P:<n> = /root/reference/PAPER.md line n; S:<x> = SURVEY.md §8(c) item x)
 *   O0  Verlet pair set  { (i,j), i<j : d2(i,j) < (rcut+skin)^2 }              P:53 "list L_i of all the
 *       particles inside a sphere centred on i of radius r_v = r_c + r_s";  S:O0 fixes the arithmetic.
 *   O1  Lennard-Jones, Eq. (1), cut and shifted at r_c  P:99.
 *   O2  WCA = O1 cut at 2^(1/6) sigma, shifted by +eps (BASELINE.json config C3/C4).
 *   O3  FENE bonds along linear chains (config C3).
 *   O4  Patchy rigid bodies of config C4: WCA core + 16-term patch-patch sum, forces and torques.
 *   O5  Energies U, K_trans, K_rot.
 *   O6  velocity-Verlet NVE (BASELINE.json north_star "md_integrate velocity-Verlet").
 *   O7  rigid-body velocity-Verlet for a spherical top (S:O7).
 *   O8  the paper's own patchy model (S:8(f2)): Eq. (3) core (sigma/r)^200 plus Eq. (4) patch-patch terms
 *       -eps exp[-1/2 (r^{ij}/0.12 sigma)^n] over the M x M patch pairs, r^{ij} the distance between patch i of
 *       particle 1 and patch j of particle 2.  Eq. (4) is garbled in PAPER.md (no minus sign, n undefined) and
 *       the patch positions are not stated: reading S:Q1 (n = 10, patches on the surface at 0.5 sigma, antipodal
 *       for M = 2, r_c = 0.18 sigma cuts r^{ij}).  PARITY UNPINNED for that reading (the cited sources are not in
 *       the container); the arithmetic of the reading itself is pinned (closed forms, finite differences,
 *       Newton-3 invariants).
 *   O9  the NVT thermostat of P:53 (Ref. 27, not in the container): reading DESIGN.md QT, an Andersen-type
 *       velocity refresh driven by Philox4x32-10.  PARITY UNPINNED with respect to Ref. 27; the reading's
 *       arithmetic is pinned (see O9 below).
 *   O10 the same sums as O1-O5 accumulated the way a CPU MD code does it: ONE thread walks the half Verlet list
 *       (i < j) once and applies Newton's third law to both members ("single CPU core").  It exists only
 *       as the single-core timing baseline of S:8(d); pinned against the plain definition (brute force), the fcc
 *       lattice sums and sum F = 0.
 * Forces/torques/energies are the PLAIN DEFINITION: a direct sum over all pairs with d2 < rcut^2
 * (both strategies evaluate exactly the pairs of the Verlet list that are inside r_c).
 * The oracle's own cell list only prunes pairs that cannot be inside the cutoff; `use_cells=0`
 * runs the O(N^2) double loop and the two are compared in tests (pins P6/P8).
 *
 * Arithmetic: IEEE fp64, compile with -ffp-contract=off (no FMA contraction), inputs are the same
 * fp32 arrays the GPU gets, converted exactly to double.  Fixed operation order for d2 (S:O0):
 *   dx = xj - xi; if (dx > 0.5*Lx) dx -= Lx; else if (dx < -0.5*Lx) dx += Lx;   (same y, z)
 *   d2 = (dx*dx + dy*dy) + dz*dz;   inside = d2 < rv*rv  (strict)
 *
 * Parity pins (tests/test_oracle_pins.py): closed forms P1-P4, fcc lattice sums P5, brute force P6/P8,
 * Newton-3 invariants P7, finite-difference force/torque vs energy, NVE drift P9, free rotor P10,
 * Fig. 1 thread counts P12.  Only O8 (patch_point_pair) and O9 (thermostat) are "parity unpinned"
 * (see O8 above, O9 below).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { ORC_LJ = 0, ORC_FENE_WCA = 1, ORC_PATCHY = 2, ORC_PATCHY_PP = 3 };

typedef struct {
    int kind;
    double epsilon, sigma, mass;
    double rcut;          /* outer cutoff: LJ r_c; FENE_WCA: 2^(1/6) sigma; PATCHY: patch cutoff 1.5 sigma */
    int shift_energy;     /* LJ: subtract V(rcut) */
    double fene_K, fene_R0;
    int chain_len;
    int n_patches;
    double patch_dir[8][3];
    double eps_patch, patch_sigma_r, patch_sigma_ang;
    double rcut_core;     /* PATCHY: WCA core cut 2^(1/6) sigma */
    double inertia;
    /* ORC_PATCHY_PP (O8, the paper's own patchy model, Eqs. (2)-(4) P:103-113, reading S:Q1) */
    double patch_radius;  /* distance of a patch from the centre of its particle (0.5 sigma, S:Q1)            */
    double patch_exponent;/* n of Eq. (4) (10, S:Q1)                                                          */
    double core_exponent; /* 200 of Eq. (3)                                                                   */
    double rcut_patch;    /* cut on the patch-patch distance r^{ij} (0.18 sigma); rcut = 2 patch_radius + rcut_patch */
} orc_pot;

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---- S:O0 minimum image and squared distance, fixed operation order ---- */
static inline double min_image(double d, double L) {
    if (d > 0.5 * L) d -= L;
    else if (d < -0.5 * L) d += L;
    return d;
}

static inline double dist2(const double* xi, const double* xj, const double* box, double* rvec) {
    double dx = min_image(xj[0] - xi[0], box[0]);
    double dy = min_image(xj[1] - xi[1], box[1]);
    double dz = min_image(xj[2] - xi[2], box[2]);
    rvec[0] = dx; rvec[1] = dy; rvec[2] = dz;
    return (dx * dx + dy * dy) + dz * dz;
}

/* ---- the oracle's own cell list (S:Q8): n_k = max(1, floor(L_k / (r (1+1e-5)))) ---- */
typedef struct {
    int n[3];
    int64_t ncell;
    int64_t* start;   /* ncell+1 */
    int64_t* items;   /* N, particle ids sorted by cell, ascending id inside a cell */
} cell_list;

static int cell_coord(double x, double L, int n) {
    double w = x - L * floor(x / L);        /* wrap into [0,L) for binning only */
    int c = (int)floor(w / L * n);
    if (c >= n) c = n - 1;
    if (c < 0) c = 0;
    return c;
}

static void cells_build(cell_list* cl, int64_t N, const double* pos, const double* box, double r) {
    for (int k = 0; k < 3; ++k) {
        int n = (int)floor(box[k] / (r * (1.0 + 1e-5)));
        cl->n[k] = n < 1 ? 1 : n;
    }
    cl->ncell = (int64_t)cl->n[0] * cl->n[1] * cl->n[2];
    cl->start = (int64_t*)calloc((size_t)cl->ncell + 1, sizeof(int64_t));
    cl->items = (int64_t*)malloc((size_t)(N > 0 ? N : 1) * sizeof(int64_t));
    int64_t* cof = (int64_t*)malloc((size_t)(N > 0 ? N : 1) * sizeof(int64_t));
    for (int64_t i = 0; i < N; ++i) {
        int cx = cell_coord(pos[3 * i + 0], box[0], cl->n[0]);
        int cy = cell_coord(pos[3 * i + 1], box[1], cl->n[1]);
        int cz = cell_coord(pos[3 * i + 2], box[2], cl->n[2]);
        cof[i] = ((int64_t)cx * cl->n[1] + cy) * cl->n[2] + cz;
        cl->start[cof[i] + 1]++;
    }
    for (int64_t c = 0; c < cl->ncell; ++c) cl->start[c + 1] += cl->start[c];
    int64_t* fill = (int64_t*)malloc((size_t)cl->ncell * sizeof(int64_t));
    memcpy(fill, cl->start, (size_t)cl->ncell * sizeof(int64_t));
    for (int64_t i = 0; i < N; ++i) cl->items[fill[cof[i]]++] = i;
    free(fill);
    free(cof);
}

static void cells_free(cell_list* cl) { free(cl->start); free(cl->items); }

/* distinct neighbour cells of the cell holding x (27-stencil, de-duplicated when n_k < 3) */
static int cells_stencil(const cell_list* cl, const double* x, const double* box, int64_t* out) {
    int c[3], cnt[3], lst[3][3];
    for (int k = 0; k < 3; ++k) {
        c[k] = cell_coord(x[k], box[k], cl->n[k]);
        int n = cl->n[k];
        if (n == 1) { cnt[k] = 1; lst[k][0] = 0; }
        else if (n == 2) { cnt[k] = 2; lst[k][0] = 0; lst[k][1] = 1; }
        else { cnt[k] = 3; lst[k][0] = (c[k] + n - 1) % n; lst[k][1] = c[k]; lst[k][2] = (c[k] + 1) % n; }
    }
    int m = 0;
    for (int a = 0; a < cnt[0]; ++a)
        for (int b = 0; b < cnt[1]; ++b)
            for (int d = 0; d < cnt[2]; ++d)
                out[m++] = ((int64_t)lst[0][a] * cl->n[1] + lst[1][b]) * cl->n[2] + lst[2][d];
    return m;
}

static double* to_double(const float* a, int64_t n) {
    double* d = (double*)malloc((size_t)(n > 0 ? n : 1) * sizeof(double));
    for (int64_t i = 0; i < n; ++i) d[i] = (double)a[i];
    return d;
}

/* =====================================================================================
 * O0 -- Verlet pair set.  Returns the number of pairs; writes min(count, cap) pairs
 * (i<j, original ids) sorted lexicographically into pairs[2*k], pairs[2*k+1].
 * ===================================================================================== */
static int cmp_i64(const void* a, const void* b) {
    int64_t x = *(const int64_t*)a, y = *(const int64_t*)b;
    return (x > y) - (x < y);
}

int64_t orc_pair_set_d(int64_t N, const double* pos, const double* box, double rv, int use_cells,
                       int32_t* pairs, int64_t cap) {
    const double rv2 = rv * rv;
    int64_t total = 0;
    double rvec[3];
    if (!use_cells) {
        for (int64_t i = 0; i < N; ++i)
            for (int64_t j = i + 1; j < N; ++j)
                if (dist2(pos + 3 * i, pos + 3 * j, box, rvec) < rv2) {
                    if (total < cap) { pairs[2 * total] = (int32_t)i; pairs[2 * total + 1] = (int32_t)j; }
                    ++total;
                }
        return total;
    }
    cell_list cl;
    cells_build(&cl, N, pos, box, rv);
    int64_t tmpcap = 1024;
    int64_t* tmp = (int64_t*)malloc((size_t)tmpcap * sizeof(int64_t));
    for (int64_t i = 0; i < N; ++i) {
        int64_t nb[27];
        int m = cells_stencil(&cl, pos + 3 * i, box, nb);
        int64_t cnt = 0;
        for (int s = 0; s < m; ++s)
            for (int64_t t = cl.start[nb[s]]; t < cl.start[nb[s] + 1]; ++t) {
                int64_t j = cl.items[t];
                if (j <= i) continue;
                if (dist2(pos + 3 * i, pos + 3 * j, box, rvec) < rv2) {
                    if (cnt == tmpcap) { tmpcap *= 2; tmp = (int64_t*)realloc(tmp, (size_t)tmpcap * sizeof(int64_t)); }
                    tmp[cnt++] = j;
                }
            }
        qsort(tmp, (size_t)cnt, sizeof(int64_t), cmp_i64);
        for (int64_t k = 0; k < cnt; ++k) {
            if (total < cap) { pairs[2 * total] = (int32_t)i; pairs[2 * total + 1] = (int32_t)tmp[k]; }
            ++total;
        }
    }
    free(tmp);
    cells_free(&cl);
    return total;
}

int64_t orc_pair_set(int64_t N, const float* pos3, const double* box, double rcut, double skin, int use_cells,
                     int32_t* pairs, int64_t cap) {
    double* pos = to_double(pos3, 3 * N);
    int64_t n = orc_pair_set_d(N, pos, box, rcut + skin, use_cells, pairs, cap);
    free(pos);
    return n;
}

/* =====================================================================================
 * Pair functions.  Convention (S:O1): r_vec = r_j - r_i; the force on j is +g*r_vec, on i -g*r_vec,
 * so positive g = repulsion.  Each returns the pair energy V and writes dV/dr_vec (gradient with
 * respect to r_vec): F_j = -dVdr, F_i = +dVdr.
 * ===================================================================================== */

/* O1, Eq. (1):  V = 4 eps [ (sigma/r)^12 - (sigma/r)^6 ] - V_c,  V_c = V_LJ(rcut) if shifted.
 * Energy shift only; the force is unmodified (S:Q2). */
static double lj_pair(double d2, const double* rvec, double eps, double sigma, double rcut, int shift, double* dVdr) {
    double s2 = sigma * sigma / d2;
    double s6 = s2 * s2 * s2;
    double V = 4.0 * eps * s6 * (s6 - 1.0);
    if (shift) {
        double c2 = sigma * sigma / (rcut * rcut);
        double c6 = c2 * c2 * c2;
        V -= 4.0 * eps * c6 * (c6 - 1.0);
    }
    double g = 24.0 * eps * s6 * (2.0 * s6 - 1.0) / d2;   /* -(1/r) dV/dr */
    dVdr[0] = -g * rvec[0]; dVdr[1] = -g * rvec[1]; dVdr[2] = -g * rvec[2];
    return V;
}

/* O3 FENE: U_b = -1/2 K R0^2 ln(1 - d2/R0^2); dU/dr_vec = K r_vec / (1 - d2/R0^2) */
static double fene_pair(double d2, const double* rvec, double K, double R0, double* dVdr, int* bad) {
    double q = 1.0 - d2 / (R0 * R0);
    if (!(q > 0.0)) { *bad = 1; dVdr[0] = dVdr[1] = dVdr[2] = 0.0; return 0.0; }
    double c = K / q;
    dVdr[0] = c * rvec[0]; dVdr[1] = c * rvec[1]; dVdr[2] = c * rvec[2];
    return -0.5 * K * R0 * R0 * log(q);
}

/* rotation matrix of a unit quaternion (w,x,y,z), S:O4 */
static void quat_to_R(const double* q, double R[3][3]) {
    double w = q[0], x = q[1], y = q[2], z = q[3];
    R[0][0] = 1 - 2 * (y * y + z * z); R[0][1] = 2 * (x * y - w * z);     R[0][2] = 2 * (x * z + w * y);
    R[1][0] = 2 * (x * y + w * z);     R[1][1] = 1 - 2 * (x * x + z * z); R[1][2] = 2 * (y * z - w * x);
    R[2][0] = 2 * (x * z - w * y);     R[2][1] = 2 * (y * z + w * x);     R[2][2] = 1 - 2 * (x * x + y * y);
}

static void cross3(const double* a, const double* b, double* c) {
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}

/* O4 patch-patch term of config C4 (BASELINE.json configs[3]), the plain 16-term double sum:
 *   V_pp = - eps_p * G(r) * sum_a sum_b exp(-(1-cos th_i^a)/w^2) exp(-(1-cos th_j^b)/w^2)
 *   G(r) = exp(-(r-sigma)^2 / (2 sr^2)),  cos th_i^a = p_i^a . u,  cos th_j^b = - p_j^b . u,  u = r_vec/r.
 * Outputs dV/dr_vec, and the torques on i and on j (space frame). */
static double patch_pair(double d2, const double* rvec, const double* qi, const double* qj, const orc_pot* p,
                         double* dVdr, double* tau_i, double* tau_j) {
    double r = sqrt(d2);
    double u[3] = { rvec[0] / r, rvec[1] / r, rvec[2] / r };
    double Ri[3][3], Rj[3][3];
    quat_to_R(qi, Ri);
    quat_to_R(qj, Rj);
    double w2 = p->patch_sigma_ang * p->patch_sigma_ang;
    double sr2 = p->patch_sigma_r * p->patch_sigma_r;
    double G = exp(-(r - p->sigma) * (r - p->sigma) / (2.0 * sr2));
    double dG = -(r - p->sigma) / sr2 * G;                 /* dG/dr */
    double V = 0.0;
    dVdr[0] = dVdr[1] = dVdr[2] = 0.0;
    tau_i[0] = tau_i[1] = tau_i[2] = 0.0;
    tau_j[0] = tau_j[1] = tau_j[2] = 0.0;
    for (int a = 0; a < p->n_patches; ++a) {
        double pa[3];
        for (int k = 0; k < 3; ++k)
            pa[k] = Ri[k][0] * p->patch_dir[a][0] + Ri[k][1] * p->patch_dir[a][1] + Ri[k][2] * p->patch_dir[a][2];
        double ca = pa[0] * u[0] + pa[1] * u[1] + pa[2] * u[2];          /* cos theta_i^a */
        double ea = exp(-(1.0 - ca) / w2);
        for (int b = 0; b < p->n_patches; ++b) {
            double pb[3];
            for (int k = 0; k < 3; ++k)
                pb[k] = Rj[k][0] * p->patch_dir[b][0] + Rj[k][1] * p->patch_dir[b][1] + Rj[k][2] * p->patch_dir[b][2];
            double cb = -(pb[0] * u[0] + pb[1] * u[1] + pb[2] * u[2]);   /* cos theta_j^b */
            double eb = exp(-(1.0 - cb) / w2);
            double term = -p->eps_patch * G * ea * eb;                  /* this patch pair's energy */
            V += term;
            /* d(term)/d r_vec = term * [ (dG/G) u + (1/w2) d(ca)/dr_vec + (1/w2) d(cb)/dr_vec ]
             * d(ca)/dr_vec = (pa - ca u)/r ;  d(cb)/dr_vec = -(pb - (pb.u) u)/r = -(pb + cb u)/r */
            for (int k = 0; k < 3; ++k) {
                double dca = (pa[k] - ca * u[k]) / r;
                double dcb = -(pb[k] + cb * u[k]) / r;
                dVdr[k] += term * (dG / G * u[k] + (dca + dcb) / w2);
            }
            /* torque on i: -dV/d(rotation of i) = -(dterm/dca) (pa x u), dterm/dca = term / w2 */
            double x1[3], x2[3];
            cross3(pa, u, x1);
            for (int k = 0; k < 3; ++k) tau_i[k] += -(term / w2) * x1[k];
            /* torque on j: cb = -pb.u -> -(dterm/dcb) (pb x (-u)) */
            double mu[3] = { -u[0], -u[1], -u[2] };
            cross3(pb, mu, x2);
            for (int k = 0; k < 3; ++k) tau_j[k] += -(term / w2) * x2[k];
        }
    }
    return V;
}

/* O8, Eqs. (2)-(4) P:103-113 under reading S:Q1.  p_a = patch_radius * R_i dir_a, d = r_vec + p_b - p_a is the
 * vector from patch a of i to patch b of j, u = |d|; a patch pair contributes only if u < rcut_patch:
 *   term = -eps_patch exp(-g),  g = 1/2 (u / w)^n,   d term / d d_vec = -term n g d / u^2
 * The force on j's patch is -d term/d d_vec, on i's patch +d term/d d_vec; torques are p x F. */
static double patch_point_pair(double d2, const double* rvec, const double* qi, const double* qj, const orc_pot* p,
                               double* dVdr, double* tau_i, double* tau_j) {
    double Ri[3][3], Rj[3][3];
    quat_to_R(qi, Ri);
    quat_to_R(qj, Rj);
    /* Eq. (3): V_CM = eps (sigma/r)^m, dV/dr_vec = -m V r_vec / r^2 */
    double V = p->epsilon * pow(p->sigma * p->sigma / d2, 0.5 * p->core_exponent);
    for (int k = 0; k < 3; ++k) dVdr[k] = -p->core_exponent * V / d2 * rvec[k];
    tau_i[0] = tau_i[1] = tau_i[2] = 0.0;
    tau_j[0] = tau_j[1] = tau_j[2] = 0.0;
    for (int a = 0; a < p->n_patches; ++a) {
        double pa[3];
        for (int k = 0; k < 3; ++k)
            pa[k] = p->patch_radius * (Ri[k][0] * p->patch_dir[a][0] + Ri[k][1] * p->patch_dir[a][1] + Ri[k][2] * p->patch_dir[a][2]);
        for (int b = 0; b < p->n_patches; ++b) {
            double pb[3], d[3];
            for (int k = 0; k < 3; ++k)
                pb[k] = p->patch_radius * (Rj[k][0] * p->patch_dir[b][0] + Rj[k][1] * p->patch_dir[b][1] + Rj[k][2] * p->patch_dir[b][2]);
            for (int k = 0; k < 3; ++k) d[k] = (rvec[k] + pb[k]) - pa[k];
            double u2 = (d[0] * d[0] + d[1] * d[1]) + d[2] * d[2];
            if (!(u2 < p->rcut_patch * p->rcut_patch)) continue;
            double u = sqrt(u2);
            double g = 0.5 * pow(u / p->patch_sigma_r, p->patch_exponent);
            double term = -p->eps_patch * exp(-g);                       /* Eq. (4), one (i, j) patch pair */
            V += term;
            if (u2 > 0.0) {
                double c = -term * p->patch_exponent * g / u2;           /* d term / d d_vec = c d */
                double gd[3] = { c * d[0], c * d[1], c * d[2] }, x[3];
                for (int k = 0; k < 3; ++k) dVdr[k] += gd[k];
                cross3(pa, gd, x);                                       /* force on i's patch = +gd */
                for (int k = 0; k < 3; ++k) tau_i[k] += x[k];
                cross3(pb, gd, x);                                       /* force on j's patch = -gd */
                for (int k = 0; k < 3; ++k) tau_j[k] -= x[k];
            }
        }
    }
    return V;
}

/* One ordered pair (i <- j): energy V of the pair, gradient dV/dr_vec, torque on i.  Returns 1 if the pair
 * is inside the interaction cutoff (S:Q5: the "force can be non-zero" test is d2 < rcut^2, strict). */
static int pair_eval(const orc_pot* p, double d2, const double* rvec, const double* qi, const double* qj,
                     double* V, double* dVdr, double* tau_i, double* tau_j) {
    *V = 0.0;
    dVdr[0] = dVdr[1] = dVdr[2] = 0.0;
    tau_i[0] = tau_i[1] = tau_i[2] = 0.0;
    tau_j[0] = tau_j[1] = tau_j[2] = 0.0;
    if (!(d2 < p->rcut * p->rcut)) return 0;
    if (p->kind == ORC_LJ) {
        *V = lj_pair(d2, rvec, p->epsilon, p->sigma, p->rcut, p->shift_energy, dVdr);
    } else if (p->kind == ORC_FENE_WCA) {
        /* O2: rcut = 2^(1/6) sigma, shift = +eps */
        *V = lj_pair(d2, rvec, p->epsilon, p->sigma, p->rcut, 1, dVdr);
    } else if (p->kind == ORC_PATCHY_PP) {
        *V = patch_point_pair(d2, rvec, qi, qj, p, dVdr, tau_i, tau_j);   /* truncated, not shifted */
    } else {
        double g[3], t1[3], t2[3];
        *V = patch_pair(d2, rvec, qi, qj, p, dVdr, tau_i, tau_j);   /* truncated, not shifted (S:Q15) */
        (void)t1; (void)t2;
        if (d2 < p->rcut_core * p->rcut_core) {
            *V += lj_pair(d2, rvec, p->epsilon, p->sigma, p->rcut_core, 1, g);
            dVdr[0] += g[0]; dVdr[1] += g[1]; dVdr[2] += g[2];
        }
    }
    return 1;
}

/* =====================================================================================
 * O1-O5: forces F[N][3], torques T[N][3] (may be NULL), per-particle potential energy pe[N]
 * (half of every pair energy and half of every bond energy), all fp64.
 * Returns 0, or 1 if a FENE bond reached R0 (the GPU path reports MD_ERR_NUMERIC there).
 * n_in_cut receives the number of unordered pairs inside the interaction cutoff.
 * ===================================================================================== */
int orc_forces_d(int64_t N, const double* pos, const double* quat, const double* box, const orc_pot* p,
                 int use_cells, double* F, double* T, double* pe, int64_t* n_in_cut) {
    cell_list cl;
    if (use_cells) cells_build(&cl, N, pos, box, p->rcut);
    int64_t in_cut = 0;
    int bad = 0;
    static const double qid[4] = { 1.0, 0.0, 0.0, 0.0 };
#pragma omp parallel for schedule(dynamic, 256) reduction(+ : in_cut) reduction(| : bad)
    for (int64_t i = 0; i < N; ++i) {
        double f[3] = { 0, 0, 0 }, t[3] = { 0, 0, 0 }, e = 0.0;
        const double* qi = quat ? quat + 4 * i : qid;
        int64_t nb[27];
        int m = 1;
        if (use_cells) m = cells_stencil(&cl, pos + 3 * i, box, nb);
        for (int s = 0; s < m; ++s) {
            int64_t t0 = use_cells ? cl.start[nb[s]] : 0;
            int64_t t1 = use_cells ? cl.start[nb[s] + 1] : N;
            for (int64_t tt = t0; tt < t1; ++tt) {
                int64_t j = use_cells ? cl.items[tt] : tt;
                if (j == i) continue;
                double rvec[3], V, dVdr[3], ti[3], tj[3];
                double d2 = dist2(pos + 3 * i, pos + 3 * j, box, rvec);
                const double* qj = quat ? quat + 4 * j : qid;
                if (pair_eval(p, d2, rvec, qi, qj, &V, dVdr, ti, tj)) {
                    f[0] += dVdr[0]; f[1] += dVdr[1]; f[2] += dVdr[2];   /* F_i = +dV/dr_vec */
                    t[0] += ti[0]; t[1] += ti[1]; t[2] += ti[2];
                    e += 0.5 * V;
                    if (j > i) ++in_cut;
                }
            }
        }
        if (p->kind == ORC_FENE_WCA) {
            /* O3: static bonds (i, i+1) inside a chain, independent of any neighbour list (S:Q14) */
            int64_t partner[2] = { -1, -1 };
            if (i % p->chain_len != 0) partner[0] = i - 1;
            if ((i + 1) % p->chain_len != 0 && i + 1 < N) partner[1] = i + 1;
            for (int k = 0; k < 2; ++k) {
                int64_t j = partner[k];
                if (j < 0) continue;
                double rvec[3], dVdr[3];
                double d2 = dist2(pos + 3 * i, pos + 3 * j, box, rvec);
                int b = 0;
                double V = fene_pair(d2, rvec, p->fene_K, p->fene_R0, dVdr, &b);
                bad |= b;
                f[0] += dVdr[0]; f[1] += dVdr[1]; f[2] += dVdr[2];
                e += 0.5 * V;
            }
        }
        F[3 * i + 0] = f[0]; F[3 * i + 1] = f[1]; F[3 * i + 2] = f[2];
        if (T) { T[3 * i + 0] = t[0]; T[3 * i + 1] = t[1]; T[3 * i + 2] = t[2]; }
        pe[i] = e;
    }
    if (use_cells) cells_free(&cl);
    if (n_in_cut) *n_in_cut = in_cut;
    return bad;
}

int orc_forces(int64_t N, const float* pos3, const float* quat4, const double* box, const orc_pot* p,
               int use_cells, double* F, double* T, double* pe, int64_t* n_in_cut) {
    double* pos = to_double(pos3, 3 * N);
    double* quat = quat4 ? to_double(quat4, 4 * N) : NULL;
    int rc = orc_forces_d(N, pos, quat, box, p, use_cells, F, T, pe, n_in_cut);
    free(pos);
    free(quat);
    return rc;
}

/* O10 (S:8(d) "single-threaded over its own half pair list with Newton's third law (the classic CPU inner loop)",
 * P:41): pairs = the half Verlet list O0 (i < j, npairs rows of two ids).  Every listed pair is evaluated
 * once; F_i += dV/dr_vec, F_j -= dV/dr_vec, half the pair energy to each, torques to each.  Bonds (O3) are walked
 * once per bond (i, i+1).  Single-threaded by construction.  Same return value as orc_forces_d. */
int orc_forces_half_d(int64_t N, const double* pos, const double* quat, const double* box, const orc_pot* p,
                      const int32_t* pairs, int64_t npairs, double* F, double* T, double* pe, int64_t* n_in_cut) {
    static const double qid[4] = { 1.0, 0.0, 0.0, 0.0 };
    int64_t in_cut = 0;
    int bad = 0;
    memset(F, 0, sizeof(double) * 3 * (size_t)N);
    if (T) memset(T, 0, sizeof(double) * 3 * (size_t)N);
    memset(pe, 0, sizeof(double) * (size_t)N);
    for (int64_t e = 0; e < npairs; ++e) {
        const int64_t i = pairs[2 * e], j = pairs[2 * e + 1];
        double rvec[3], V, dVdr[3], ti[3], tj[3];
        const double d2 = dist2(pos + 3 * i, pos + 3 * j, box, rvec);
        const double* qi = quat ? quat + 4 * i : qid;
        const double* qj = quat ? quat + 4 * j : qid;
        if (!pair_eval(p, d2, rvec, qi, qj, &V, dVdr, ti, tj)) continue;
        ++in_cut;
        for (int k = 0; k < 3; ++k) { F[3 * i + k] += dVdr[k]; F[3 * j + k] -= dVdr[k]; }   /* F_i = +dV/dr_vec = -F_j */
        if (T) for (int k = 0; k < 3; ++k) { T[3 * i + k] += ti[k]; T[3 * j + k] += tj[k]; }
        pe[i] += 0.5 * V; pe[j] += 0.5 * V;
    }
    if (p->kind == ORC_FENE_WCA) {
        for (int64_t i = 0; i + 1 < N; ++i) {
            if ((i + 1) % p->chain_len == 0) continue;
            double rvec[3], dVdr[3];
            const double d2 = dist2(pos + 3 * i, pos + 3 * (i + 1), box, rvec);
            int b = 0;
            const double V = fene_pair(d2, rvec, p->fene_K, p->fene_R0, dVdr, &b);
            bad |= b;
            for (int k = 0; k < 3; ++k) { F[3 * i + k] += dVdr[k]; F[3 * (i + 1) + k] -= dVdr[k]; }
            pe[i] += 0.5 * V; pe[i + 1] += 0.5 * V;
        }
    }
    if (n_in_cut) *n_in_cut = in_cut;
    return bad;
}

int orc_forces_half(int64_t N, const float* pos3, const float* quat4, const double* box, const orc_pot* p,
                    const int32_t* pairs, int64_t npairs, double* F, double* T, double* pe, int64_t* n_in_cut) {
    double* pos = to_double(pos3, 3 * N);
    double* quat = quat4 ? to_double(quat4, 4 * N) : NULL;
    int rc = orc_forces_half_d(N, pos, quat, box, p, pairs, npairs, F, T, pe, n_in_cut);
    free(pos);
    free(quat);
    return rc;
}

/* One unordered pair evaluated in isolation (used by the closed-form pins and by the pair invariant
 * tau_i + tau_j + r_vec x F_j = 0, pin P7).  rvec = r_j - r_i given directly, no periodic box. */
int orc_pair(const orc_pot* p, const double* rvec, const double* qi, const double* qj,
             double* V, double* F_j, double* tau_i, double* tau_j) {
    double d2 = (rvec[0] * rvec[0] + rvec[1] * rvec[1]) + rvec[2] * rvec[2];
    double dVdr[3];
    int in = pair_eval(p, d2, rvec, qi, qj, V, dVdr, tau_i, tau_j);
    F_j[0] = -dVdr[0]; F_j[1] = -dVdr[1]; F_j[2] = -dVdr[2];
    return in;
}

/* FENE bond in isolation */
int orc_bond(const orc_pot* p, const double* rvec, double* V, double* F_j) {
    double d2 = (rvec[0] * rvec[0] + rvec[1] * rvec[1]) + rvec[2] * rvec[2];
    double dVdr[3];
    int bad = 0;
    *V = fene_pair(d2, rvec, p->fene_K, p->fene_R0, dVdr, &bad);
    F_j[0] = -dVdr[0]; F_j[1] = -dVdr[1]; F_j[2] = -dVdr[2];
    return bad;
}

/* O5 */
void orc_energy_d(int64_t N, const double* pe, const double* vel, const double* angmom, double mass, double inertia,
                  double* U, double* Kt, double* Kr) {
    double u = 0, kt = 0, kr = 0;
    for (int64_t i = 0; i < N; ++i) {
        u += pe[i];
        kt += 0.5 * mass * ((vel[3 * i] * vel[3 * i] + vel[3 * i + 1] * vel[3 * i + 1]) + vel[3 * i + 2] * vel[3 * i + 2]);
        if (angmom)
            kr += ((angmom[3 * i] * angmom[3 * i] + angmom[3 * i + 1] * angmom[3 * i + 1]) + angmom[3 * i + 2] * angmom[3 * i + 2])
                  / (2.0 * inertia);
    }
    *U = u; *Kt = kt; *Kr = kr;
}

/* =====================================================================================
 * O6 / O7: velocity-Verlet NVE on fp64 state, step by step (S:O6, S:O7):
 *   v += dt/2 F/m ; [L += dt/2 tau ; omega = L/I ; q <- dq (x) q ; renormalise] ; x += dt v ;
 *   skin check (S:Q4): max_i |x_i - x_i^ref|^2 > (skin/2)^2 -> wrap, "rebuild", x^ref = x ;
 *   F, tau = forces(x, q) ; v += dt/2 F/m ; [L += dt/2 tau].
 * The forces do not depend on the list (plain definition), so the rebuild is book-keeping for the
 * rebuild count only.  energies[3*k..] = (U, K_t, K_r) after step (k+1)*every; F/T/pe hold the
 * forces on entry (must be valid) and on exit.
 * ===================================================================================== */
int orc_integrate_d(int64_t N, double* pos, double* vel, double* quat, double* angmom, const double* box,
                    const orc_pot* p, double skin, double dt, int64_t nsteps, int64_t every,
                    double* F, double* T, double* pe, double* energies, int64_t* n_rebuilds) {
    double* ref = (double*)malloc((size_t)(3 * N + 1) * sizeof(double));
    memcpy(ref, pos, (size_t)(3 * N) * sizeof(double));
    int64_t rebuilds = 0;
    int bad = 0;
    const double hs2 = (0.5 * skin) * (0.5 * skin);
    for (int64_t s = 0; s < nsteps; ++s) {
        for (int64_t i = 0; i < N; ++i)
            for (int k = 0; k < 3; ++k) {
                vel[3 * i + k] += 0.5 * dt * F[3 * i + k] / p->mass;
                pos[3 * i + k] += dt * vel[3 * i + k];
            }
        if (quat) {
            for (int64_t i = 0; i < N; ++i) {
                double w[3], wn;
                for (int k = 0; k < 3; ++k) {
                    angmom[3 * i + k] += 0.5 * dt * T[3 * i + k];
                    w[k] = angmom[3 * i + k] / p->inertia;
                }
                wn = sqrt((w[0] * w[0] + w[1] * w[1]) + w[2] * w[2]);
                if (wn > 0.0) {
                    double h = 0.5 * wn * dt, c = cos(h), sn = sin(h) / wn;
                    double a[4] = { c, sn * w[0], sn * w[1], sn * w[2] };   /* dq */
                    double* q = quat + 4 * i;
                    double r[4];                                         /* dq (x) q : space-frame axis */
                    r[0] = a[0] * q[0] - a[1] * q[1] - a[2] * q[2] - a[3] * q[3];
                    r[1] = a[0] * q[1] + a[1] * q[0] + a[2] * q[3] - a[3] * q[2];
                    r[2] = a[0] * q[2] - a[1] * q[3] + a[2] * q[0] + a[3] * q[1];
                    r[3] = a[0] * q[3] + a[1] * q[2] - a[2] * q[1] + a[3] * q[0];
                    double nrm = sqrt((r[0] * r[0] + r[1] * r[1]) + (r[2] * r[2] + r[3] * r[3]));
                    for (int k = 0; k < 4; ++k) q[k] = r[k] / nrm;
                }
            }
        }
        double dmax = 0.0;
        for (int64_t i = 0; i < N; ++i) {
            double d = 0;
            for (int k = 0; k < 3; ++k) { double t = pos[3 * i + k] - ref[3 * i + k]; d += t * t; }
            if (d > dmax) dmax = d;
        }
        if (dmax > hs2) {
            for (int64_t i = 0; i < 3 * N; ++i) { int k = (int)(i % 3); pos[i] -= box[k] * floor(pos[i] / box[k]); }
            memcpy(ref, pos, (size_t)(3 * N) * sizeof(double));
            ++rebuilds;
        }
        bad |= orc_forces_d(N, pos, quat, box, p, 1, F, T, pe, NULL);
        for (int64_t i = 0; i < N; ++i)
            for (int k = 0; k < 3; ++k) {
                vel[3 * i + k] += 0.5 * dt * F[3 * i + k] / p->mass;
                if (quat) angmom[3 * i + k] += 0.5 * dt * T[3 * i + k];
            }
        if (energies && every > 0 && (s + 1) % every == 0) {
            int64_t k = (s + 1) / every - 1;
            orc_energy_d(N, pe, vel, quat ? angmom : NULL, p->mass, p->inertia,
                         energies + 3 * k, energies + 3 * k + 1, energies + 3 * k + 2);
        }
    }
    free(ref);
    if (n_rebuilds) *n_rebuilds = rebuilds;
    return bad;
}

/* =====================================================================================
 * O9: the NVT thermostat the paper names but does not describe ("Brownian dynamics simulations in
 * the NVT ensemble, with the thermostat described in Ref. 27"; S:8(f3), item 12 of S:2).  Ref. 27 is not in
 * the container: reading DESIGN.md QT -- an Andersen-type velocity refresh: after every n_newt-th
 * velocity-Verlet step each particle, independently and with probability p_t, has its velocity replaced by
 * a Maxwell-Boltzmann draw at temperature T (each component Gaussian of variance k_B T / m); a rigid body,
 * with probability p_r, likewise its angular momentum (variance k_B T I).  PARITY UNPINNED with respect to
 * Ref. 27; the arithmetic of the reading is pinned (Philox known answers, moments and a KS test of the draws,
 * refreshed fraction, p = 0 and p = 1, relaxation of an LJ fluid to the target temperature).
 *
 * Random numbers: the counter-based generator Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11); both
 * sides implement it, nothing is shared.  key = (seed low word, seed high word); counter =
 * (particle id, call index, stream, block): stream 0 = translation, 1 = rotation; block 0 word 0 decides
 * (refresh iff word0 < floor(p 2^32), compared in 64 bits so that p = 1 always refreshes); block 1 words
 * 0..3 give u_k = (word_k + 0.5) 2^-32 and, by Box-Muller in fp64,
 *   g0 = sqrt(-2 ln u0) cos(2 pi u1), g1 = sqrt(-2 ln u0) sin(2 pi u1), g2 = sqrt(-2 ln u2) cos(2 pi u3).
 * ===================================================================================== */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* one stream of one particle: returns 1 and the three Gaussians if the particle is refreshed */
static int thermostat_draw(uint32_t id, uint32_t call, uint32_t stream, uint64_t seed, double p, double g[3]) {
    const uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
    uint32_t c[4] = { id, call, stream, 0u }, w[4];
    double thr_d = floor(p * 4294967296.0);
    uint64_t thr = thr_d <= 0.0 ? 0u : (thr_d >= 4294967296.0 ? 4294967296ull : (uint64_t)thr_d);
    orc_philox4x32_10(c, key, w);
    if (!((uint64_t)w[0] < thr)) return 0;
    c[3] = 1u;
    orc_philox4x32_10(c, key, w);
    const double two_pi = 6.283185307179586476925286766559;
    double u0 = ((double)w[0] + 0.5) / 4294967296.0, u1 = ((double)w[1] + 0.5) / 4294967296.0;
    double u2 = ((double)w[2] + 0.5) / 4294967296.0, u3 = ((double)w[3] + 0.5) / 4294967296.0;
    double r0 = sqrt(-2.0 * log(u0)), r1 = sqrt(-2.0 * log(u2));
    g[0] = r0 * cos(two_pi * u1);
    g[1] = r0 * sin(two_pi * u1);
    g[2] = r1 * cos(two_pi * u3);
    return 1;
}

/* one application of the thermostat to fp64 state in id order; returns the number of refreshed velocities
 * (n_rot: refreshed angular momenta).  angmom may be NULL. */
int64_t orc_thermostat_d(int64_t N, double* vel, double* angmom, double mass, double inertia, double T,
                         double p_t, double p_r, uint64_t seed, uint32_t call, int64_t* n_rot) {
    int64_t nt = 0, nr = 0;
    const double sv = sqrt(T / mass), sl = sqrt(T * inertia);
    for (int64_t i = 0; i < N; ++i) {
        double g[3];
        if (thermostat_draw((uint32_t)i, call, 0u, seed, p_t, g)) {
            for (int k = 0; k < 3; ++k) vel[3 * i + k] = sv * g[k];
            ++nt;
        }
        if (angmom && thermostat_draw((uint32_t)i, call, 1u, seed, p_r, g)) {
            for (int k = 0; k < 3; ++k) angmom[3 * i + k] = sl * g[k];
            ++nr;
        }
    }
    if (n_rot) *n_rot = nr;
    return nt;
}
