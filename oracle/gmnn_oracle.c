/*
 * gmnn_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, fp64 CPU statement of the Gaussian Moment Neural Network energy-and-force
 * evaluation of arxiv 2505.22168 (apax), written from PAPER.md Eq. 1-6 and the readings listed
 * in DESIGN.md section 3.  It is the parity reference for the CUDA path and the timed
 * `cpu_baseline` of bench.py.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.  It shares no code, header, table or helper with
 * paper_2505_22168_b200/ and is never tuned for speed: naive loops over full (un-symmetrised)
 * tensors, O(N^2 * images) neighbour search, OpenMP over atoms only so that it finishes.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): forces == central finite differences of the
 * energy; sum F = 0; E invariant under rotation / translation+wrap / permutation; brute-force ==
 * cell-list neighbour sets; dimer and simple-cubic closed forms; trace identities of the moments;
 * MLP == numpy matmul; Eq. 6 linearity of the ensemble; NVE dt^2 scaling and time reversal;
 * O-12: identical heads give sigma = 0 and the single-head NVE trajectory, the sampled trajectory does
 * not depend on sampling_rate, sigma_E against numpy's std of the head totals, stop at the first
 * sample over the threshold (tests/test_oracle_switching.py).
 * Parity unpinned by the paper itself: PAPER.md prints no numeric E or F for any geometry, and the
 * constants of DESIGN.md readings R1-R4, R7-R10 are readings, not quotes.
 *
 * Passages followed:
 *   O-1  neighbour set ............ PAPER.md:49 ("local neighbors"), :171 (several images), :381 (skin)
 *   O-2  radial functions ......... PAPER.md:49-52 (equidistant Gaussians, element-pair coefficients)
 *   O-3  moments .................. PAPER.md:51 (Eq. 2)
 *   O-4  invariants ............... PAPER.md:54-61 (Eq. 3; "up to L=3 and 4-body terms")
 *   O-5  readout + scale-shift .... PAPER.md:63-65 (Eq. 4), :151 (ensemble axis not summed)
 *   O-6  total energy ............. PAPER.md:46 (Eq. 1)
 *   O-7..O-9 forces = -dE/dR ...... PAPER.md:127, 153 (gradient of the energy), chain rule by hand
 *   O-10 ensemble ................. PAPER.md:75-88 (Eq. 5 with 1/N_ens, Eq. 6)
 *   O-11 NVE velocity Verlet ...... BASELINE.json configs 2, 5; dt PAPER.md:367; skin :381
 *   O-12 switching-mode ensemble MD  PAPER.md:175 (Eq. 6: cheap mean-energy forces every step, the
 *        per-head pass only every N steps), :71 (uncertainty as stopping criterion), Eq. 5
 *   O-13 UDD bias (gmnn_oracle.py, numpy on O-10's per-head forces)  PAPER.md:102-107 (Eq. 9); pins in
 *        tests/test_oracle_udd.py: forces == finite differences of mean + E_b, limits of Eq. 9, conservation
 *   O-14 NVT, Nose-Hoover chain (gmnn_oracle.py)  PAPER.md:365-375 (thermostat_chain keys); pins in
 *        tests/test_oracle_nvt.py: conserved extended energy at second order, tau -> inf is O-11, heating
 *        towards the target, closed form and time reversal of one chain operator
 *   O-15 Langevin, BAOAB + counter-based normals (gmnn_oracle.py)  PAPER.md:266; pins in
 *        tests/test_oracle_langevin.py: published splitmix64 value, moments and independence of the normals,
 *        gamma = 0 is O-11, gamma dt >> 1 gives E_kin = 3/2 N kT (units of the noise), relaxation to the target
 *
 * Build: gcc -O2 -std=c11 -fPIC -shared -fopenmp -ffp-contract=off gmnn_oracle.c -lm
 *        (-ffp-contract=off: the neighbour predicate is specified in unfused fp32, reading R20.)
 */
#define _GNU_SOURCE
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NC 40 /* components per radial channel: 1 (L=0) + 3 (L=1) + 9 (L=2) + 27 (L=3) */
#define O0 0
#define O1 1
#define O2 4
#define O3 13
#define ACC_CONV 9.648533212e-3 /* (eV/Ang/amu) -> Ang/fs^2 */

typedef struct {
    int32_t n_species, n_basis, n_radial;
    double r_cut, r_min, gamma;
    int32_t n_hidden;
    int32_t hidden[4];
    int32_t n_heads;
    int32_t n_weight_sets; /* 1 (or 0): one NN for all species (Eq. 4); n_species: the (W, b) of set Z_i (O-5) */
    int32_t basis_kind;    /* 0: equidistant Gaussians (O-2); 1: Bessel-like functions of Kocer et al. (O-17) */
    int32_t zbl_on;        /* 1: add the ZBL repulsion (O-18) */
    double zbl_r_max;      /* Ang, cutoff of the ZBL term (<= r_cut) */
    double zbl_scale;      /* dimensionless prefactor of the ZBL term */
} oracle_hparams;

typedef struct {
    const double *beta;  /* [S][S][n_radial][n_basis], centre species first */
    const double *W[5];  /* layer l: [n_weight_sets][fan_in][fan_out] row-major, set-major */
    const double *b[5];  /* layer l: [n_weight_sets][fan_out] */
    const double *scale; /* [S] sigma_Z */
    const double *shift; /* [S] mu_Z */
    const double *atomic_number; /* [S] nuclear charges Z (O-18), nullable when zbl_on == 0 */
} oracle_weights;

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* Feature count of O-4 (blocks 0..7). */
int oracle_n_features(int n) {
    int pairs = n * (n + 1) / 2;
    int triples = n * (n + 1) * (n + 2) / 6;
    return n + 3 * pairs + triples + 2 * pairs * n + n * n * n;
}

/* ------------------------------------------------------------------------------------------
 * O-1  Neighbour set.  r_list = r_cut + skin.  Cell h (row-major 3x3, rows = lattice vectors a, b, c;
 * O-16: any right- or left-handed lattice, the configs' boxes are diag(L)).  For every i, j and image
 * n in [-k..k]^3, k_a = pbc_a ? ceil(r_list / w_a) : 0 with w_a the distance between the two cell faces
 * that axis a connects (w_a = V / |b x c| ...; = L_a for diag(L)), excluding (j == i, n == 0):
 * keep (i, j, n) iff |x_j - x_i + n1 a + n2 b + n3 c|^2 < r_list^2, strict.  Full list (both directions).
 * Positions must lie inside the cell (fractional coordinates in [0, 1) on periodic axes).
 * The predicate is SPECIFIED in unfused fp32 (reading R20; O-16 extends the shift to three terms):
 *   s_x = fl(fl(fl(n1 a_x) + fl(n2 b_x)) + fl(n3 c_x))   (= fl(n1 L_x) for diag(L): adding a zero is exact)
 *   d_x = fl(fl(x_j,x - x_i,x) + s_x);  r2 = fl(fl(dx*dx + dy*dy) + dz*dz);  keep iff r2 < fl(r_list * r_list).
 * Output sorted by (i, j, n1, n2, n3).  Returns the number of pairs; writes at most cap of them.
 * ------------------------------------------------------------------------------------------ */
static inline int pair_predicate(const float *pos, int64_t i, int64_t j, float sx, float sy, float sz, float rl2) {
    float dx = (pos[3 * j + 0] - pos[3 * i + 0]) + sx;
    float dy = (pos[3 * j + 1] - pos[3 * i + 1]) + sy;
    float dz = (pos[3 * j + 2] - pos[3 * i + 2]) + sz;
    float r2 = (dx * dx + dy * dy) + dz * dz;
    return r2 < rl2;
}

/* fp32 lattice shift of image (n1, n2, n3), in the order the predicate fixes */
static inline void image_shift32(const float *h, int n1, int n2, int n3, float *s) {
    for (int x = 0; x < 3; ++x) s[x] = ((float)n1 * h[0 + x] + (float)n2 * h[3 + x]) + (float)n3 * h[6 + x];
}

/* distance between opposite faces of the cell along each lattice direction: w_a = V / |b x c|, ... */
static void face_distances(const double *h, double *w) {
    const double *a = h, *b = h + 3, *c = h + 6;
    double bc[3] = {b[1] * c[2] - b[2] * c[1], b[2] * c[0] - b[0] * c[2], b[0] * c[1] - b[1] * c[0]};
    double ca[3] = {c[1] * a[2] - c[2] * a[1], c[2] * a[0] - c[0] * a[2], c[0] * a[1] - c[1] * a[0]};
    double ab[3] = {a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]};
    double V = fabs(a[0] * bc[0] + a[1] * bc[1] + a[2] * bc[2]);
    w[0] = V / sqrt(bc[0] * bc[0] + bc[1] * bc[1] + bc[2] * bc[2]);
    w[1] = V / sqrt(ca[0] * ca[0] + ca[1] * ca[1] + ca[2] * ca[2]);
    w[2] = V / sqrt(ab[0] * ab[0] + ab[1] * ab[1] + ab[2] * ab[2]);
}

/* inverse of the row-major cell: fractional coordinates s = x hinv (row vector times matrix) */
static void cell_inverse(const double *h, double *hi) {
    double det = h[0] * (h[4] * h[8] - h[5] * h[7]) - h[1] * (h[3] * h[8] - h[5] * h[6]) + h[2] * (h[3] * h[7] - h[4] * h[6]);
    hi[0] = (h[4] * h[8] - h[5] * h[7]) / det;
    hi[1] = (h[2] * h[7] - h[1] * h[8]) / det;
    hi[2] = (h[1] * h[5] - h[2] * h[4]) / det;
    hi[3] = (h[5] * h[6] - h[3] * h[8]) / det;
    hi[4] = (h[0] * h[8] - h[2] * h[6]) / det;
    hi[5] = (h[2] * h[3] - h[0] * h[5]) / det;
    hi[6] = (h[3] * h[7] - h[4] * h[6]) / det;
    hi[7] = (h[1] * h[6] - h[0] * h[7]) / det;
    hi[8] = (h[0] * h[4] - h[1] * h[3]) / det;
}

static int cell_is_diagonal(const double *h) {
    return h[1] == 0.0 && h[2] == 0.0 && h[3] == 0.0 && h[5] == 0.0 && h[6] == 0.0 && h[7] == 0.0;
}

int64_t oracle_neighbors_brute(int64_t N, const float *pos, const float *h, const int32_t *pbc, float r_list,
                               int64_t cap, int32_t *out_i, int32_t *out_j, int32_t *out_n) {
    int k[3];
    double hd[9], w[3];
    for (int q = 0; q < 9; ++q) hd[q] = (double)h[q];
    face_distances(hd, w);
    for (int a = 0; a < 3; ++a) k[a] = pbc[a] ? (int)ceil((double)r_list / w[a]) : 0;
    const float rl2 = r_list * r_list;
    int64_t count = 0;
    for (int64_t i = 0; i < N; ++i)
        for (int64_t j = 0; j < N; ++j)
            for (int nx = -k[0]; nx <= k[0]; ++nx)
                for (int ny = -k[1]; ny <= k[1]; ++ny)
                    for (int nz = -k[2]; nz <= k[2]; ++nz) {
                        if (j == i && nx == 0 && ny == 0 && nz == 0) continue;
                        float sh[3];
                        image_shift32(h, nx, ny, nz, sh);
                        if (pair_predicate(pos, i, j, sh[0], sh[1], sh[2], rl2)) {
                            if (count < cap) {
                                out_i[count] = (int32_t)i;
                                out_j[count] = (int32_t)j;
                                out_n[3 * count + 0] = nx;
                                out_n[3 * count + 1] = ny;
                                out_n[3 * count + 2] = nz;
                            }
                            ++count;
                        }
                    }
    return count;
}

typedef struct {
    int32_t j, nx, ny, nz;
} cand_t;

static int cand_cmp(const void *a, const void *b) {
    const cand_t *x = (const cand_t *)a, *y = (const cand_t *)b;
    if (x->j != y->j) return x->j < y->j ? -1 : 1;
    if (x->nx != y->nx) return x->nx < y->nx ? -1 : 1;
    if (x->ny != y->ny) return x->ny < y->ny ? -1 : 1;
    if (x->nz != y->nz) return x->nz < y->nz ? -1 : 1;
    return 0;
}

/* The oracle's own O(N) search (linked cells), used for N > 8192 and itself pinned against the
 * brute force above.  Same predicate, same output order.  Needs >= 3 cells on every periodic
 * axis (else returns -1: use the brute force). */
int64_t oracle_neighbors_cells(int64_t N, const float *pos, const float *h, const int32_t *pbc, float r_list,
                               int64_t cap, int32_t *out_i, int32_t *out_j, int32_t *out_n) {
    int nc[3];
    double hd[9], hinv[9], w[3];
    for (int q = 0; q < 9; ++q) hd[q] = (double)h[q];
    face_distances(hd, w);
    cell_inverse(hd, hinv);
    for (int a = 0; a < 3; ++a) {  /* bins in fractional coordinates: slabs at least r_list thick */
        nc[a] = (int)floor(w[a] / ((double)r_list * (1.0 + 1e-6)));
        if (nc[a] < 1) nc[a] = 1;
        if (pbc[a] && nc[a] < 3) return -1;
    }
    const float rl2 = r_list * r_list;
    int64_t ncell = (int64_t)nc[0] * nc[1] * nc[2];
    int64_t *head = (int64_t *)malloc(sizeof(int64_t) * (size_t)ncell);
    int64_t *next = (int64_t *)malloc(sizeof(int64_t) * (size_t)N);
    int32_t *cidx = (int32_t *)malloc(sizeof(int32_t) * 3 * (size_t)N);
    for (int64_t c = 0; c < ncell; ++c) head[c] = -1;
    for (int64_t i = N - 1; i >= 0; --i) {
        int c[3];
        for (int a = 0; a < 3; ++a) {
            double frac = 0.0;
            for (int x = 0; x < 3; ++x) frac += (double)pos[3 * i + x] * hinv[3 * x + a];
            c[a] = (int)floor(frac * nc[a]);
            if (c[a] < 0) c[a] = 0;
            if (c[a] >= nc[a]) c[a] = nc[a] - 1;
            cidx[3 * i + a] = c[a];
        }
        int64_t cc = ((int64_t)c[0] * nc[1] + c[1]) * nc[2] + c[2];
        next[i] = head[cc];
        head[cc] = i;
    }
    int64_t count = 0;
    size_t cand_cap = 1024;
    cand_t *cand = (cand_t *)malloc(sizeof(cand_t) * cand_cap);
    for (int64_t i = 0; i < N; ++i) {
        size_t nc_i = 0;
        for (int ox = -1; ox <= 1; ++ox)
            for (int oy = -1; oy <= 1; ++oy)
                for (int oz = -1; oz <= 1; ++oz) {
                    int o[3] = {ox, oy, oz}, c[3], n[3];
                    int skip = 0;
                    for (int a = 0; a < 3; ++a) {
                        c[a] = cidx[3 * i + a] + o[a];
                        n[a] = 0;
                        if (c[a] < 0) {
                            if (!pbc[a]) { skip = 1; break; }
                            c[a] += nc[a];
                            n[a] = -1;
                        } else if (c[a] >= nc[a]) {
                            if (!pbc[a]) { skip = 1; break; }
                            c[a] -= nc[a];
                            n[a] = 1;
                        }
                    }
                    if (skip) continue;
                    /* with fewer than 3 cells on a NON-periodic axis, offsets can alias: visit once */
                    int dup = 0;
                    for (int a = 0; a < 3; ++a)
                        if (!pbc[a] && nc[a] < 3 && (cidx[3 * i + a] + o[a] < 0 || cidx[3 * i + a] + o[a] >= nc[a])) dup = 1;
                    if (dup) continue;
                    float sh[3];
                    image_shift32(h, n[0], n[1], n[2], sh);
                    int64_t cc = ((int64_t)c[0] * nc[1] + c[1]) * nc[2] + c[2];
                    for (int64_t j = head[cc]; j >= 0; j = next[j]) {
                        if (j == i && n[0] == 0 && n[1] == 0 && n[2] == 0) continue;
                        if (pair_predicate(pos, i, j, sh[0], sh[1], sh[2], rl2)) {
                            if (nc_i == cand_cap) {
                                cand_cap *= 2;
                                cand = (cand_t *)realloc(cand, sizeof(cand_t) * cand_cap);
                            }
                            cand[nc_i].j = (int32_t)j;
                            cand[nc_i].nx = n[0];
                            cand[nc_i].ny = n[1];
                            cand[nc_i].nz = n[2];
                            ++nc_i;
                        }
                    }
                }
        qsort(cand, nc_i, sizeof(cand_t), cand_cmp);
        for (size_t q = 0; q < nc_i; ++q) {
            if (count < cap) {
                out_i[count] = (int32_t)i;
                out_j[count] = cand[q].j;
                out_n[3 * count + 0] = cand[q].nx;
                out_n[3 * count + 1] = cand[q].ny;
                out_n[3 * count + 2] = cand[q].nz;
            }
            ++count;
        }
    }
    free(cand);
    free(head);
    free(next);
    free(cidx);
    return count;
}

/* ------------------------------------------------------------------------------------------
 * O-2  Radial functions of one pair (readings R1-R4).
 *   mu_k = r_min + k Delta, Delta = (r_cut - r_min)/(n_b - 1);  Phi_k = exp(-gamma (r - mu_k)^2)
 *   f_c = 1/2 [1 + cos(pi r / r_cut)]  (r < r_cut, else 0)
 *   R_s = f_c sum_k beta[Zi][Zj][s][k] Phi_k
 *   R'_s = f_c' sum_k beta Phi_k + f_c sum_k beta Phi_k (-2 gamma (r - mu_k)),
 *   f_c' = -(pi / (2 r_cut)) sin(pi r / r_cut)
 * ------------------------------------------------------------------------------------------ */
/* O-2 / O-17  The n_basis basis functions of one distance and their derivatives (no cutoff function).
 * kind 0 ("equidistant Gaussians"): Phi_k = exp(-gamma (r - mu_k)^2), mu_k = r_min + k Delta.
 * kind 1 ("the non-orthogonal Bessel-like functions of Kocer et al."; reading R30), n = 0..n_b-1:
 *   f_n(r) = (-1)^n sqrt(2) pi / r_c^(3/2) (n+1)(n+2) / sqrt((n+1)^2 + (n+2)^2)
 *            [ sinc((n+1) pi r / r_c) + sinc((n+2) pi r / r_c) ],   sinc(x) = sin(x) / x
 *   (unit norm under int_0^rc . r^2 dr; zero at r_c; the orthogonalisation step of that paper is not applied),
 *   d/dr sinc(a r) = (cos(a r) - sinc(a r)) / r. */
void oracle_basis(const oracle_hparams *hp, double r, double *phi, double *dphi) {
    const int nb = hp->n_basis;
    if (hp->basis_kind == 1) {
        const double rc = hp->r_cut;
        for (int n = 0; n < nb; ++n) {
            double a1 = (n + 1) * M_PI / rc, a2 = (n + 2) * M_PI / rc;
            double c = ((n & 1) ? -1.0 : 1.0) * sqrt(2.0) * M_PI / pow(rc, 1.5) * (n + 1.0) * (n + 2.0) /
                       sqrt((n + 1.0) * (n + 1.0) + (n + 2.0) * (n + 2.0));
            double s1 = sin(a1 * r) / (a1 * r), s2 = sin(a2 * r) / (a2 * r);
            phi[n] = c * (s1 + s2);
            if (dphi) dphi[n] = c * ((cos(a1 * r) - s1) + (cos(a2 * r) - s2)) / r;
        }
        return;
    }
    const double delta = (hp->r_cut - hp->r_min) / (nb - 1);
    for (int k = 0; k < nb; ++k) {
        double mu = hp->r_min + k * delta;
        phi[k] = exp(-hp->gamma * (r - mu) * (r - mu));
        if (dphi) dphi[k] = phi[k] * (-2.0 * hp->gamma * (r - mu));
    }
}

void oracle_radial(const oracle_hparams *hp, const double *beta, int zi, int zj, double r, double *R, double *dR) {
    const int nb = hp->n_basis, nr = hp->n_radial, S = hp->n_species;
    if (r >= hp->r_cut) {
        for (int s = 0; s < nr; ++s) {
            R[s] = 0.0;
            if (dR) dR[s] = 0.0;
        }
        return;
    }
    double phi[64], dphi[64];
    oracle_basis(hp, r, phi, dphi);
    const double fc = 0.5 * (1.0 + cos(M_PI * r / hp->r_cut));
    const double dfc = -0.5 * M_PI / hp->r_cut * sin(M_PI * r / hp->r_cut);
    for (int s = 0; s < nr; ++s) {
        double sum = 0.0, dsum = 0.0;
        for (int k = 0; k < nb; ++k) {
            double bk = beta[(((size_t)zi * S + zj) * nr + s) * nb + k];
            sum += bk * phi[k];
            dsum += bk * dphi[k];
        }
        R[s] = fc * sum;
        if (dR) dR[s] = dfc * sum + fc * dsum;
    }
}

/* ------------------------------------------------------------------------------------------
 * O-18  ZBL repulsion ("empirical energy correction terms, such as the Ziegler-Littmark-Biersack
 * potential, can be supplied"; reading R31).  For a pair of nuclear charges Z1, Z2 at distance r < r_zbl:
 *   V(r) = scale k_e Z1 Z2 / r  phi(r / a)  f_c(r; r_zbl),   k_e = 14.399645 eV Ang,
 *   a = 0.8854 a_0 / (Z1^0.23 + Z2^0.23),  a_0 = 0.529177 Ang,
 *   phi(x) = 0.1818 e^(-3.2 x) + 0.5099 e^(-0.9423 x) + 0.2802 e^(-0.4029 x) + 0.02817 e^(-0.2016 x),
 *   f_c = 1/2 [1 + cos(pi r / r_zbl)].
 * E gets V once per unordered pair: every DIRECTED pair of the full list carries V/2, added to the centre's E_i
 * (after sigma, mu: it is not a network output).  Returns V/2 and d(V/2)/dr.
 * ------------------------------------------------------------------------------------------ */
void oracle_zbl_half(const oracle_hparams *hp, double z1, double z2, double r, double *e, double *de) {
    *e = 0.0;
    if (de) *de = 0.0;
    if (!hp->zbl_on || r >= hp->zbl_r_max) return;
    static const double c[4] = {0.1818, 0.5099, 0.2802, 0.02817}, d[4] = {3.2, 0.9423, 0.4029, 0.2016};
    const double a = 0.8854 * 0.529177 / (pow(z1, 0.23) + pow(z2, 0.23));
    double phi = 0.0, dphi = 0.0;
    for (int k = 0; k < 4; ++k) {
        phi += c[k] * exp(-d[k] * r / a);
        dphi += c[k] * exp(-d[k] * r / a) * (-d[k] / a);
    }
    const double coul = 0.5 * hp->zbl_scale * 14.399645 * z1 * z2 / r, dcoul = -coul / r;
    const double fc = 0.5 * (1.0 + cos(M_PI * r / hp->zbl_r_max));
    const double dfc = -0.5 * M_PI / hp->zbl_r_max * sin(M_PI * r / hp->zbl_r_max);
    *e = coul * phi * fc;
    if (de) *de = dcoul * phi * fc + coul * dphi * fc + coul * phi * dfc;
}

/* d = x_j - x_i + n1 a + n2 b + n3 c in fp64 (positions are fp32 values promoted to fp64; L = the 3x3 cell, rows a, b, c). */
static inline void pair_vector(const double *pos, const double *L, int64_t i, int64_t j, const int32_t *n, double *d) {
    for (int x = 0; x < 3; ++x)
        d[x] = pos[3 * j + x] - pos[3 * i + x] + (n[0] * L[0 + x] + n[1] * L[3 + x] + n[2] * L[6 + x]);
}

/* ------------------------------------------------------------------------------------------
 * O-3  Moments of one atom (Eq. 2): u = d / r (direction i -> j);
 *   P0[s] += R_s;  P1[s]_a += R_s u_a;  P2[s]_ab += R_s u_a u_b;  P3[s]_abc += R_s u_a u_b u_c.
 * P is [n_radial][NC] with offsets O0, O1 + a, O2 + 3a + b, O3 + 9a + 3b + c.
 * Pairs in the skin shell (r >= r_cut) contribute nothing.
 * ------------------------------------------------------------------------------------------ */
static void moments_of_atom(const oracle_hparams *hp, const double *beta, const double *pos, const int32_t *species,
                            const double *L, int64_t i, int64_t p_begin, int64_t p_end, const int32_t *pj,
                            const int32_t *pn, double *P) {
    const int nr = hp->n_radial;
    double R[16];
    memset(P, 0, sizeof(double) * (size_t)nr * NC);
    for (int64_t p = p_begin; p < p_end; ++p) {
        double d[3];
        pair_vector(pos, L, i, pj[p], pn + 3 * p, d);
        double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        if (r >= hp->r_cut) continue;
        double u[3] = {d[0] / r, d[1] / r, d[2] / r};
        oracle_radial(hp, beta, species[i], species[pj[p]], r, R, NULL);
        for (int s = 0; s < nr; ++s) {
            double *Ps = P + (size_t)s * NC;
            Ps[O0] += R[s];
            for (int a = 0; a < 3; ++a) {
                Ps[O1 + a] += R[s] * u[a];
                for (int b = 0; b < 3; ++b) {
                    Ps[O2 + 3 * a + b] += R[s] * u[a] * u[b];
                    for (int c = 0; c < 3; ++c) Ps[O3 + 9 * a + 3 * b + c] += R[s] * u[a] * u[b] * u[c];
                }
            }
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * O-4  Invariants (Eq. 3).  First printed line = block 1, last printed line = block 7; the
 * elided middle is completed with every full contraction of <= 3 moments with L <= 3 that is not
 * a product of smaller ones (reading R7).  Blocks concatenated in this order; inside a block the
 * index tuples run in lexicographic order and only symmetry-unique tuples are kept (R8):
 *   0: P0[s]                                      s
 *   1: P1[s1]_a   P1[s2]_a                        s1 <= s2
 *   2: P2[s1]_ab  P2[s2]_ab                       s1 <= s2
 *   3: P3[s1]_abc P3[s2]_abc                      s1 <= s2
 *   4: P2[s1]_ab  P2[s2]_bc  P2[s3]_ca            s1 <= s2 <= s3
 *   5: P1[s1]_a   P1[s2]_b   P2[s3]_ab            s1 <= s2, all s3
 *   6: P3[s1]_abc P3[s2]_abd P2[s3]_cd            s1 <= s2, all s3
 *   7: P1[s1]_a   P3[s2]_abc P2[s3]_bc            all s1, s2, s3
 * ------------------------------------------------------------------------------------------ */
#define P1_(s, a) P[(size_t)(s) * NC + O1 + (a)]
#define P2_(s, a, b) P[(size_t)(s) * NC + O2 + 3 * (a) + (b)]
#define P3_(s, a, b, c) P[(size_t)(s) * NC + O3 + 9 * (a) + 3 * (b) + (c)]
#define Q1_(s, a) Q[(size_t)(s) * NC + O1 + (a)]
#define Q2_(s, a, b) Q[(size_t)(s) * NC + O2 + 3 * (a) + (b)]
#define Q3_(s, a, b, c) Q[(size_t)(s) * NC + O3 + 9 * (a) + 3 * (b) + (c)]

void oracle_invariants(int nr, const double *P, double *G) {
    int f = 0;
    for (int s = 0; s < nr; ++s) G[f++] = P[(size_t)s * NC + O0];
    for (int s1 = 0; s1 < nr; ++s1)
        for (int s2 = s1; s2 < nr; ++s2) {
            double g = 0.0;
            for (int a = 0; a < 3; ++a) g += P1_(s1, a) * P1_(s2, a);
            G[f++] = g;
        }
    for (int s1 = 0; s1 < nr; ++s1)
        for (int s2 = s1; s2 < nr; ++s2) {
            double g = 0.0;
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b) g += P2_(s1, a, b) * P2_(s2, a, b);
            G[f++] = g;
        }
    for (int s1 = 0; s1 < nr; ++s1)
        for (int s2 = s1; s2 < nr; ++s2) {
            double g = 0.0;
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b)
                    for (int c = 0; c < 3; ++c) g += P3_(s1, a, b, c) * P3_(s2, a, b, c);
            G[f++] = g;
        }
    for (int s1 = 0; s1 < nr; ++s1)
        for (int s2 = s1; s2 < nr; ++s2)
            for (int s3 = s2; s3 < nr; ++s3) {
                double g = 0.0;
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b)
                        for (int c = 0; c < 3; ++c) g += P2_(s1, a, b) * P2_(s2, b, c) * P2_(s3, c, a);
                G[f++] = g;
            }
    for (int s1 = 0; s1 < nr; ++s1)
        for (int s2 = s1; s2 < nr; ++s2)
            for (int s3 = 0; s3 < nr; ++s3) {
                double g = 0.0;
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b) g += P1_(s1, a) * P1_(s2, b) * P2_(s3, a, b);
                G[f++] = g;
            }
    for (int s1 = 0; s1 < nr; ++s1)
        for (int s2 = s1; s2 < nr; ++s2)
            for (int s3 = 0; s3 < nr; ++s3) {
                double g = 0.0;
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b)
                        for (int c = 0; c < 3; ++c)
                            for (int d = 0; d < 3; ++d) g += P3_(s1, a, b, c) * P3_(s2, a, b, d) * P2_(s3, c, d);
                G[f++] = g;
            }
    for (int s1 = 0; s1 < nr; ++s1)
        for (int s2 = 0; s2 < nr; ++s2)
            for (int s3 = 0; s3 < nr; ++s3) {
                double g = 0.0;
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b)
                        for (int c = 0; c < 3; ++c) g += P1_(s1, a) * P3_(s2, a, b, c) * P2_(s3, b, c);
                G[f++] = g;
            }
}

/* ------------------------------------------------------------------------------------------
 * O-8  Backward of O-4: Q = dE/dP given gb = dE/dG, every one of the 1+3+9+27 entries per
 * channel treated as independent; a contribution is added for EACH slot even when channel
 * indices coincide.  Q2, Q3 come out non-symmetric; that is intended.
 * ------------------------------------------------------------------------------------------ */
void oracle_invariants_bwd(int nr, const double *P, const double *gb, double *Q) {
    memset(Q, 0, sizeof(double) * (size_t)nr * NC);
    int f = 0;
    for (int s = 0; s < nr; ++s) Q[(size_t)s * NC + O0] += gb[f++];
    for (int s1 = 0; s1 < nr; ++s1)
        for (int s2 = s1; s2 < nr; ++s2) {
            double g = gb[f++];
            for (int a = 0; a < 3; ++a) {
                Q1_(s1, a) += g * P1_(s2, a);
                Q1_(s2, a) += g * P1_(s1, a);
            }
        }
    for (int s1 = 0; s1 < nr; ++s1)
        for (int s2 = s1; s2 < nr; ++s2) {
            double g = gb[f++];
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b) {
                    Q2_(s1, a, b) += g * P2_(s2, a, b);
                    Q2_(s2, a, b) += g * P2_(s1, a, b);
                }
        }
    for (int s1 = 0; s1 < nr; ++s1)
        for (int s2 = s1; s2 < nr; ++s2) {
            double g = gb[f++];
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b)
                    for (int c = 0; c < 3; ++c) {
                        Q3_(s1, a, b, c) += g * P3_(s2, a, b, c);
                        Q3_(s2, a, b, c) += g * P3_(s1, a, b, c);
                    }
        }
    for (int s1 = 0; s1 < nr; ++s1)
        for (int s2 = s1; s2 < nr; ++s2)
            for (int s3 = s2; s3 < nr; ++s3) {
                double g = gb[f++];
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b)
                        for (int c = 0; c < 3; ++c) {
                            /* term = P2[s1]_ab P2[s2]_bc P2[s3]_ca */
                            Q2_(s1, a, b) += g * P2_(s2, b, c) * P2_(s3, c, a);
                            Q2_(s2, b, c) += g * P2_(s1, a, b) * P2_(s3, c, a);
                            Q2_(s3, c, a) += g * P2_(s1, a, b) * P2_(s2, b, c);
                        }
            }
    for (int s1 = 0; s1 < nr; ++s1)
        for (int s2 = s1; s2 < nr; ++s2)
            for (int s3 = 0; s3 < nr; ++s3) {
                double g = gb[f++];
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b) {
                        /* term = P1[s1]_a P1[s2]_b P2[s3]_ab */
                        Q1_(s1, a) += g * P1_(s2, b) * P2_(s3, a, b);
                        Q1_(s2, b) += g * P1_(s1, a) * P2_(s3, a, b);
                        Q2_(s3, a, b) += g * P1_(s1, a) * P1_(s2, b);
                    }
            }
    for (int s1 = 0; s1 < nr; ++s1)
        for (int s2 = s1; s2 < nr; ++s2)
            for (int s3 = 0; s3 < nr; ++s3) {
                double g = gb[f++];
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b)
                        for (int c = 0; c < 3; ++c)
                            for (int d = 0; d < 3; ++d) {
                                /* term = P3[s1]_abc P3[s2]_abd P2[s3]_cd */
                                Q3_(s1, a, b, c) += g * P3_(s2, a, b, d) * P2_(s3, c, d);
                                Q3_(s2, a, b, d) += g * P3_(s1, a, b, c) * P2_(s3, c, d);
                                Q2_(s3, c, d) += g * P3_(s1, a, b, c) * P3_(s2, a, b, d);
                            }
            }
    for (int s1 = 0; s1 < nr; ++s1)
        for (int s2 = 0; s2 < nr; ++s2)
            for (int s3 = 0; s3 < nr; ++s3) {
                double g = gb[f++];
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b)
                        for (int c = 0; c < 3; ++c) {
                            /* term = P1[s1]_a P3[s2]_abc P2[s3]_bc */
                            Q1_(s1, a) += g * P3_(s2, a, b, c) * P2_(s3, b, c);
                            Q3_(s2, a, b, c) += g * P1_(s1, a) * P2_(s3, b, c);
                            Q2_(s3, b, c) += g * P1_(s1, a) * P3_(s2, a, b, c);
                        }
            }
}

/* ------------------------------------------------------------------------------------------
 * O-5  Readout (Eq. 4): z1 = G W1 + b1; h1 = swish(z1); ...; y = h W_last + b_last
 * in R^M.  swish(x) = x sigmoid(x) (reading R10).  zs holds the pre-activations of the hidden
 * layers back to back (sum of hidden[] doubles).  Eq. 4 prints one NN for all species (n_weight_sets
 * = 1, set 0); with n_weight_sets = n_species ("the per-species atomic MLP", reading R11) atom i uses
 * the (W, b) of set Z_i.  Pins: tests/test_oracle_species_mlp.py.
 * ------------------------------------------------------------------------------------------ */
static inline double sigmoid_(double x) { return 1.0 / (1.0 + exp(-x)); }
static inline double swish_(double x) { return x * sigmoid_(x); }
static inline double dswish_(double x) {
    double s = sigmoid_(x);
    return s * (1.0 + x * (1.0 - s));
}
double oracle_swish(double x) { return swish_(x); }
double oracle_dswish(double x) { return dswish_(x); }

/* Weights of layer l for weight set `wset` (0 when the NN is shared): O-5, "the (W, b) used are those of set Z_i". */
static const double *layer_W(const oracle_hparams *hp, const oracle_weights *w, int n_in, int l, int wset) {
    int fi = l > 0 ? hp->hidden[l - 1] : n_in;
    int fo = l < hp->n_hidden ? hp->hidden[l] : hp->n_heads;
    return w->W[l] + (size_t)wset * fi * fo;
}
static const double *layer_b(const oracle_hparams *hp, const oracle_weights *w, int l, int wset) {
    int fo = l < hp->n_hidden ? hp->hidden[l] : hp->n_heads;
    return w->b[l] + (size_t)wset * fo;
}
/* Which weight set atom of species z uses. */
static int weight_set_of(const oracle_hparams *hp, int z) { return hp->n_weight_sets > 1 ? z : 0; }

void oracle_mlp_forward(const oracle_hparams *hp, const oracle_weights *w, int n_in, const double *G, double *zs,
                        double *y, int wset) {
    const double *h = G;
    int fan_in = n_in;
    double hbuf[2][4096];
    double *z = zs;
    for (int l = 0; l < hp->n_hidden; ++l) {
        int fo = hp->hidden[l];
        const double *Wl = layer_W(hp, w, n_in, l, wset), *bl = layer_b(hp, w, l, wset);
        for (int o = 0; o < fo; ++o) {
            double acc = bl[o];
            for (int k = 0; k < fan_in; ++k) acc += h[k] * Wl[(size_t)k * fo + o];
            z[o] = acc;
        }
        double *hn = hbuf[l & 1];
        for (int o = 0; o < fo; ++o) hn[o] = swish_(z[o]);
        h = hn;
        z += fo;
        fan_in = fo;
    }
    const int L = hp->n_hidden, M = hp->n_heads;
    const double *WL = layer_W(hp, w, n_in, L, wset), *bL = layer_b(hp, w, L, wset);
    for (int m = 0; m < M; ++m) {
        double acc = bL[m];
        for (int k = 0; k < fan_in; ++k) acc += h[k] * WL[(size_t)k * M + m];
        y[m] = acc;
    }
}

/* O-7  Backward to the features: ybar[m] given; hbar = W_last ybar; zbar = hbar * swish'(z);
 * ... ; Gbar = W1 zbar1. */
void oracle_mlp_backward(const oracle_hparams *hp, const oracle_weights *w, int n_in, const double *zs,
                         const double *ybar, double *Gbar, int wset) {
    const int L = hp->n_hidden, M = hp->n_heads;
    double buf[2][4096];
    int width_last = L > 0 ? hp->hidden[L - 1] : n_in;
    double *hb = buf[0];
    const double *WL = layer_W(hp, w, n_in, L, wset);
    for (int k = 0; k < width_last; ++k) {
        double acc = 0.0;
        for (int m = 0; m < M; ++m) acc += WL[(size_t)k * M + m] * ybar[m];
        hb[k] = acc;
    }
    int zoff = 0;
    for (int l = 0; l < L; ++l) zoff += hp->hidden[l];
    for (int l = L - 1; l >= 0; --l) {
        int fo = hp->hidden[l];
        int fi = l > 0 ? hp->hidden[l - 1] : n_in;
        zoff -= fo;
        const double *z = zs + zoff;
        double *nb = buf[(L - l) & 1];
        const double *Wl = layer_W(hp, w, n_in, l, wset);
        for (int k = 0; k < fi; ++k) nb[k] = 0.0;
        for (int o = 0; o < fo; ++o) {
            double zb = hb[o] * dswish_(z[o]);
            for (int k = 0; k < fi; ++k) nb[k] += Wl[(size_t)k * fo + o] * zb;
        }
        hb = nb;
    }
    for (int k = 0; k < n_in; ++k) Gbar[k] = hb[k];
}

/* ------------------------------------------------------------------------------------------
 * O-9  Pair gradient for one kept pair with r < r_cut, using Q of the centre atom i:
 *   c_s = Q0[s] + Q1[s]_a u_a + Q2[s]_ab u_a u_b + Q3[s]_abc u_a u_b u_c
 *   w_a = sum_s R_s [ Q1[s]_a + (Q2[s]_ab + Q2[s]_ba) u_b
 *                     + (Q3[s]_abc + Q3[s]_bac + Q3[s]_bca) u_b u_c ]
 *   g   = (sum_s R'_s c_s) u + (w - (w.u) u) / r        ( = dE/dd )
 * F_i += g;  F_j -= g   (d = x_j - x_i + shift, so dE/dx_i = -g and F = -dE/dx).
 * ------------------------------------------------------------------------------------------ */
static void pair_gradient(const oracle_hparams *hp, const double *beta, int zi, int zj, const double *d,
                          const double *Q, double *g) {
    const int nr = hp->n_radial;
    double R[16], dR[16];
    double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    g[0] = g[1] = g[2] = 0.0;
    if (r >= hp->r_cut) return;
    double u[3] = {d[0] / r, d[1] / r, d[2] / r};
    oracle_radial(hp, beta, zi, zj, r, R, dR);
    double radial = 0.0, w[3] = {0.0, 0.0, 0.0};
    for (int s = 0; s < nr; ++s) {
        double c = Q[(size_t)s * NC + O0];
        for (int a = 0; a < 3; ++a) {
            c += Q1_(s, a) * u[a];
            for (int b = 0; b < 3; ++b) {
                c += Q2_(s, a, b) * u[a] * u[b];
                for (int cc = 0; cc < 3; ++cc) c += Q3_(s, a, b, cc) * u[a] * u[b] * u[cc];
            }
        }
        radial += dR[s] * c;
        for (int a = 0; a < 3; ++a) {
            double t = Q1_(s, a);
            for (int b = 0; b < 3; ++b) {
                t += (Q2_(s, a, b) + Q2_(s, b, a)) * u[b];
                for (int cc = 0; cc < 3; ++cc)
                    t += (Q3_(s, a, b, cc) + Q3_(s, b, a, cc) + Q3_(s, b, cc, a)) * u[b] * u[cc];
            }
            w[a] += R[s] * t;
        }
    }
    double wu = w[0] * u[0] + w[1] * u[1] + w[2] * u[2];
    for (int a = 0; a < 3; ++a) g[a] = radial * u[a] + (w[a] - wu * u[a]) / r;
}

/* CSR row offsets of a pair list sorted by i. */
static int64_t *row_offsets(int64_t N, int64_t npairs, const int32_t *pi) {
    int64_t *off = (int64_t *)calloc((size_t)N + 1, sizeof(int64_t));
    for (int64_t p = 0; p < npairs; ++p) off[pi[p] + 1]++;
    for (int64_t i = 0; i < N; ++i) off[i + 1] += off[i];
    return off;
}

static int total_hidden(const oracle_hparams *hp) {
    int t = 0;
    for (int l = 0; l < hp->n_hidden; ++l) t += hp->hidden[l];
    return t;
}

/* Forward of every atom: P [N][nr][NC], G [N][F], zs [N][sum hidden], E_heads [N][M]
 * (E_i^(m) = sigma[Z_i] y_m + mu[Z_i], reading R12). */
static void forward_all(const oracle_hparams *hp, const oracle_weights *w, int64_t N, const double *pos,
                        const int32_t *species, const double *L, const int64_t *off, const int32_t *pj,
                        const int32_t *pn, double *P, double *G, double *zs, double *E_heads) {
    const int nr = hp->n_radial, F = oracle_n_features(nr), H = total_hidden(hp), M = hp->n_heads;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t i = 0; i < N; ++i) {
        double y[64];
        double *Pi = P + (size_t)i * nr * NC;
        moments_of_atom(hp, w->beta, pos, species, L, i, off[i], off[i + 1], pj, pn, Pi);
        oracle_invariants(nr, Pi, G + (size_t)i * F);
        oracle_mlp_forward(hp, w, F, G + (size_t)i * F, zs + (size_t)i * H, y, weight_set_of(hp, species[i]));
        double ezbl = 0.0;  /* O-18: half of every pair's ZBL energy, all directed pairs of the centre */
        if (hp->zbl_on)
            for (int64_t p = off[i]; p < off[i + 1]; ++p) {
                double d[3], e;
                pair_vector(pos, L, i, pj[p], pn + 3 * p, d);
                oracle_zbl_half(hp, w->atomic_number[species[i]], w->atomic_number[species[pj[p]]],
                                sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]), &e, NULL);
                ezbl += e;
            }
        for (int m = 0; m < M; ++m) E_heads[(size_t)i * M + m] = w->scale[species[i]] * y[m] + w->shift[species[i]] + ezbl;
    }
}

/* Backward of the energy E_c = sum_i sum_m head_w[m] E_i^(m): forces [N][3]; optional dG, Q. */
static void backward_all(const oracle_hparams *hp, const oracle_weights *w, int64_t N, const double *pos,
                         const int32_t *species, const double *L, int64_t npairs, const int64_t *off,
                         const int32_t *pj, const int32_t *pn, const double *P, const double *zs,
                         const double *head_w, double *Fout, double *dG_out, double *Q_out, double *virial_out) {
    const int nr = hp->n_radial, F = oracle_n_features(nr), H = total_hidden(hp), M = hp->n_heads;
    double *gpair = (double *)malloc(sizeof(double) * 3 * (size_t)(npairs > 0 ? npairs : 1));
    memset(Fout, 0, sizeof(double) * 3 * (size_t)N);
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t i = 0; i < N; ++i) {
        double ybar[64], Gbar[1024], Qloc[16 * NC];
        for (int m = 0; m < M; ++m) ybar[m] = w->scale[species[i]] * head_w[m];
        oracle_mlp_backward(hp, w, F, zs + (size_t)i * H, ybar, Gbar, weight_set_of(hp, species[i]));
        oracle_invariants_bwd(nr, P + (size_t)i * nr * NC, Gbar, Qloc);
        if (dG_out) memcpy(dG_out + (size_t)i * F, Gbar, sizeof(double) * F);
        if (Q_out) memcpy(Q_out + (size_t)i * nr * NC, Qloc, sizeof(double) * nr * NC);
        double hw_sum = 0.0;  /* every head's energy carries the ZBL term once (O-18) */
        for (int m = 0; m < M; ++m) hw_sum += head_w[m];
        for (int64_t p = off[i]; p < off[i + 1]; ++p) {
            double d[3];
            pair_vector(pos, L, i, pj[p], pn + 3 * p, d);
            pair_gradient(hp, w->beta, species[i], species[pj[p]], d, Qloc, gpair + 3 * p);
            if (hp->zbl_on) {
                double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]), e, de;
                oracle_zbl_half(hp, w->atomic_number[species[i]], w->atomic_number[species[pj[p]]], r, &e, &de);
                for (int a = 0; a < 3; ++a) gpair[3 * p + a] += hw_sum * de * d[a] / r;
            }
            for (int a = 0; a < 3; ++a) Fout[3 * i + a] += gpair[3 * p + a];
        }
    }
    for (int64_t i = 0; i < N; ++i)
        for (int64_t p = off[i]; p < off[i + 1]; ++p)
            for (int a = 0; a < 3; ++a) Fout[3 * (size_t)pj[p] + a] -= gpair[3 * p + a];
    /* O-16  Virial ("the gradient of the energy with respect to ... the strain tensor"): under a
     * homogeneous strain d -> (1 + eps) d of every pair vector, dE/d eps_ab = sum_pairs g_a d_b with g = dE/dd
     * of the directed pair (O-9).  W_ab = - sum_pairs d_a g_b = -dE/d eps (symmetric for a rotation-invariant
     * E, which the pins check rather than assume); stress = -W / V. */
    if (virial_out) {
        for (int q = 0; q < 9; ++q) virial_out[q] = 0.0;
        for (int64_t i = 0; i < N; ++i)
            for (int64_t p = off[i]; p < off[i + 1]; ++p) {
                double d[3];
                pair_vector(pos, L, i, pj[p], pn + 3 * p, d);
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b) virial_out[3 * a + b] -= d[a] * gpair[3 * p + b];
            }
    }
    free(gpair);
}

/* ------------------------------------------------------------------------------------------
 * O-1..O-9 on a given pair list (sorted by i).  head_w[M]: weights of the heads in the energy
 * whose gradient becomes F (single model: M = 1, head_w = {1}; mean energy: 1/M each).
 * Outputs: E_heads [N][M]; F [N][3]; nullable P [N][nr][40], G [N][F], dG [N][F], Q [N][nr][40].
 * Returns 0, or -1 on a bad argument.
 * ------------------------------------------------------------------------------------------ */
int oracle_energy_forces(const oracle_hparams *hp, const oracle_weights *w, int64_t N, const double *pos,
                         const int32_t *species, const double *L, int64_t npairs, const int32_t *pi,
                         const int32_t *pj, const int32_t *pn, const double *head_w, double *E_heads, double *Fout,
                         double *P_out, double *G_out, double *dG_out, double *Q_out, double *virial_out) {
    if (hp->n_radial > 16 || hp->n_heads > 64 || hp->n_hidden > 4) return -1;
    if (hp->n_weight_sets > 1 && hp->n_weight_sets != hp->n_species) return -1;
    const int nr = hp->n_radial, F = oracle_n_features(nr), H = total_hidden(hp);
    if (F > 1024) return -1;
    for (int l = 0; l < hp->n_hidden; ++l)
        if (hp->hidden[l] > 4096) return -1;
    int64_t *off = row_offsets(N, npairs, pi);
    double *P = P_out ? P_out : (double *)malloc(sizeof(double) * (size_t)N * nr * NC);
    double *G = G_out ? G_out : (double *)malloc(sizeof(double) * (size_t)N * F);
    double *zs = (double *)malloc(sizeof(double) * (size_t)N * (H > 0 ? H : 1));
    forward_all(hp, w, N, pos, species, L, off, pj, pn, P, G, zs, E_heads);
    if (Fout) backward_all(hp, w, N, pos, species, L, npairs, off, pj, pn, P, zs, head_w, Fout, dG_out, Q_out, virial_out);
    free(off);
    if (!P_out) free(P);
    if (!G_out) free(G);
    free(zs);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O-10  Shallow ensemble (Eq. 5, 6): forward once; for every head m the backward with
 * ybar = sigma e_m gives F^(m).  e_mean_i = 1/M sum_m E_i^(m); e_var_i = 1/M sum_m (E_i^(m) -
 * mean)^2 (population divisor, reading R13); f_mean, f_var likewise per atom and component.
 * F_heads [M][N][3] nullable.
 * ------------------------------------------------------------------------------------------ */
int oracle_ensemble(const oracle_hparams *hp, const oracle_weights *w, int64_t N, const double *pos,
                    const int32_t *species, const double *L, int64_t npairs, const int32_t *pi, const int32_t *pj,
                    const int32_t *pn, double *E_heads, double *e_mean, double *e_var, double *f_mean, double *f_var,
                    double *F_heads) {
    if (hp->n_radial > 16 || hp->n_heads > 64 || hp->n_hidden > 4) return -1;
    const int nr = hp->n_radial, F = oracle_n_features(nr), H = total_hidden(hp), M = hp->n_heads;
    int64_t *off = row_offsets(N, npairs, pi);
    double *P = (double *)malloc(sizeof(double) * (size_t)N * nr * NC);
    double *G = (double *)malloc(sizeof(double) * (size_t)N * F);
    double *zs = (double *)malloc(sizeof(double) * (size_t)N * (H > 0 ? H : 1));
    double *Fall = F_heads ? F_heads : (double *)malloc(sizeof(double) * (size_t)M * N * 3);
    forward_all(hp, w, N, pos, species, L, off, pj, pn, P, G, zs, E_heads);
    for (int m = 0; m < M; ++m) {
        double hw[64];
        for (int q = 0; q < M; ++q) hw[q] = (q == m) ? 1.0 : 0.0;
        backward_all(hp, w, N, pos, species, L, npairs, off, pj, pn, P, zs, hw, Fall + (size_t)m * N * 3, NULL, NULL, NULL);
    }
    for (int64_t i = 0; i < N; ++i) {
        double mean = 0.0, var = 0.0;
        for (int m = 0; m < M; ++m) mean += E_heads[(size_t)i * M + m];
        mean /= M;
        for (int m = 0; m < M; ++m) var += (E_heads[(size_t)i * M + m] - mean) * (E_heads[(size_t)i * M + m] - mean);
        e_mean[i] = mean;
        e_var[i] = var / M;
        for (int a = 0; a < 3; ++a) {
            double fm = 0.0, fv = 0.0;
            for (int m = 0; m < M; ++m) fm += Fall[((size_t)m * N + i) * 3 + a];
            fm /= M;
            for (int m = 0; m < M; ++m) {
                double dlt = Fall[((size_t)m * N + i) * 3 + a] - fm;
                fv += dlt * dlt;
            }
            f_mean[3 * i + a] = fm;
            f_var[3 * i + a] = fv / M;
        }
    }
    free(off);
    free(P);
    free(G);
    free(zs);
    if (!F_heads) free(Fall);
    return 0;
}

/* Fold one position into the cell along the periodic axes.  diag(L): x_a -= floor(x_a / L_a) L_a;
 * general lattice (O-16): fractional s = x hinv, x -= floor(s_a) (lattice vector a). */
static void wrap_position(double *x, const double *L, const int32_t *pbc) {
    if (cell_is_diagonal(L)) {
        for (int a = 0; a < 3; ++a)
            if (pbc[a]) x[a] -= floor(x[a] / L[4 * a]) * L[4 * a];
        return;
    }
    double hinv[9];
    cell_inverse(L, hinv);
    for (int a = 0; a < 3; ++a) {
        if (!pbc[a]) continue;
        double frac = x[0] * hinv[a] + x[1] * hinv[3 + a] + x[2] * hinv[6 + a];
        double k = floor(frac);
        for (int c = 0; c < 3; ++c) x[c] -= k * L[3 * a + c];
    }
}

/* Neighbour list of fp64 positions (cast to fp32 for the predicate), growing buffers. */
typedef struct {
    int64_t n, cap;
    int32_t *i, *j, *n3;
} pairlist_t;

static void build_list(pairlist_t *pl, int64_t N, const double *pos, const double *L, const int32_t *pbc,
                       double r_list) {
    float *p32 = (float *)malloc(sizeof(float) * 3 * (size_t)N);
    float L32[9];
    for (int q = 0; q < 9; ++q) L32[q] = (float)L[q];
    for (int64_t q = 0; q < 3 * N; ++q) p32[q] = (float)pos[q];
    for (;;) {
        int64_t n = oracle_neighbors_cells(N, p32, L32, pbc, (float)r_list, pl->cap, pl->i, pl->j, pl->n3);
        if (n < 0) n = oracle_neighbors_brute(N, p32, L32, pbc, (float)r_list, pl->cap, pl->i, pl->j, pl->n3);
        if (n <= pl->cap) {
            pl->n = n;
            break;
        }
        pl->cap = n + n / 8 + 64;
        pl->i = (int32_t *)realloc(pl->i, sizeof(int32_t) * (size_t)pl->cap);
        pl->j = (int32_t *)realloc(pl->j, sizeof(int32_t) * (size_t)pl->cap);
        pl->n3 = (int32_t *)realloc(pl->n3, sizeof(int32_t) * 3 * (size_t)pl->cap);
    }
    free(p32);
}

/* ------------------------------------------------------------------------------------------
 * O-11  NVE velocity Verlet, n_steps steps of dt (fs):
 *   v += (dt/2) a(F);  x += dt v;  wrap x into [0, L) on periodic axes;
 *   if max_i |x_i - x_ref,i| > skin/2 (unwrapped displacement since the last build): rebuild,
 *   x_ref <- x;   F <- O-1..O-9;   v += (dt/2) a(F).      a = F/m * 9.648533212e-3.
 * E_kin = 1/2 sum m v^2 / 9.648533212e-3.  epot/ekin [n_steps + 1] (index 0 = initial state).
 * x, v are updated in place; x is returned wrapped.
 *
 * The image vectors n of a list refer to the coordinates it was built from, so between builds
 * the pair vectors are taken from xu, the unwrapped continuation of the build coordinates
 * (xu = x_ref + displacement); the wrapped x is xu folded back into the cell.  E and F do not
 * depend on which image of an atom is used, so this is O-11 exactly.  With skin == 0 any motion
 * exceeds skin/2 and the list is rebuilt every step.
 * ------------------------------------------------------------------------------------------ */
int oracle_nve(const oracle_hparams *hp, const oracle_weights *w, int64_t N, double *x, double *v,
               const double *masses, const int32_t *species, const double *L, const int32_t *pbc, double skin,
               double dt, int64_t n_steps, double *epot, double *ekin, int64_t *n_rebuilds) {
    if (hp->n_heads != 1) return -1;
    pairlist_t pl = {0, 0, NULL, NULL, NULL};
    double *F = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    double *Ei = (double *)malloc(sizeof(double) * (size_t)N);
    double *xu = (double *)malloc(sizeof(double) * 3 * (size_t)N);   /* list-consistent coordinates */
    double *xref = (double *)malloc(sizeof(double) * 3 * (size_t)N); /* xu at the last build */
    const double one = 1.0;
    int64_t rebuilds = 0;
    for (int64_t i = 0; i < N; ++i) wrap_position(x + 3 * i, L, pbc);
    memcpy(xu, x, sizeof(double) * 3 * (size_t)N);
    memcpy(xref, x, sizeof(double) * 3 * (size_t)N);
    build_list(&pl, N, x, L, pbc, hp->r_cut + skin);
    oracle_energy_forces(hp, w, N, xu, species, L, pl.n, pl.i, pl.j, pl.n3, &one, Ei, F, NULL, NULL, NULL, NULL, NULL);
    for (int64_t step = 0;; ++step) {
        double ep = 0.0, ek = 0.0;
        for (int64_t i = 0; i < N; ++i) {
            ep += Ei[i];
            ek += 0.5 * masses[i] * (v[3 * i] * v[3 * i] + v[3 * i + 1] * v[3 * i + 1] + v[3 * i + 2] * v[3 * i + 2]);
        }
        epot[step] = ep;
        ekin[step] = ek / ACC_CONV;
        if (step == n_steps) break;
        double maxd2 = 0.0;
        for (int64_t i = 0; i < N; ++i) {
            double d2 = 0.0;
            for (int a = 0; a < 3; ++a) {
                v[3 * i + a] += 0.5 * dt * F[3 * i + a] / masses[i] * ACC_CONV;
                xu[3 * i + a] += dt * v[3 * i + a];
                x[3 * i + a] = xu[3 * i + a];
                double dd = xu[3 * i + a] - xref[3 * i + a];
                d2 += dd * dd;
            }
            wrap_position(x + 3 * i, L, pbc);
            if (d2 > maxd2) maxd2 = d2;
        }
        if (sqrt(maxd2) > 0.5 * skin) {
            memcpy(xu, x, sizeof(double) * 3 * (size_t)N);
            memcpy(xref, x, sizeof(double) * 3 * (size_t)N);
            build_list(&pl, N, x, L, pbc, hp->r_cut + skin);
            ++rebuilds;
        }
        oracle_energy_forces(hp, w, N, xu, species, L, pl.n, pl.i, pl.j, pl.n3, &one, Ei, F, NULL, NULL, NULL, NULL, NULL);
        for (int64_t i = 0; i < N; ++i)
            for (int a = 0; a < 3; ++a) v[3 * i + a] += 0.5 * dt * F[3 * i + a] / masses[i] * ACC_CONV;
    }
    if (n_rebuilds) *n_rebuilds = rebuilds;
    free(F);
    free(Ei);
    free(xu);
    free(xref);
    free(pl.i);
    free(pl.j);
    free(pl.n3);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O-12  Switching-mode shallow-ensemble MD ("switch between the two modes during a
 * simulation ... the more expensive force uncertainty evaluation is only performed every N steps";
 * stopping criterion PAPER.md:71; Eq. 5, 6).  The loop is O-11 on the MEAN energy
 * E = 1/M sum_m E^(m) (left-hand side of Eq. 6: head weights 1/M in the backward pass).  After
 * every sampling_rate-th step (k = 1, 2, ...: after step k * sampling_rate, reading R25) the full
 * ensemble pass O-10 at the current coordinates gives (Eq. 5, divisor 1/N_ens, reading R13)
 *   sigma_e[k-1]     = sqrt(1/M sum_m (E^(m) - mean)^2),   E^(m) = sum_i E_i^(m)   (total energy)
 *   sigma_f_max[k-1] = max_i sqrt(sum_a f_var[i][a])        (Eq. 5 for x = F_i, "implied sum over
 *                      components"; the worst atom decides, reading R26)
 * and the run ends after that sample if f_sigma_stop > 0 and sigma_f_max[k-1] > f_sigma_stop.
 * epot/ekin [n_steps + 1] valid up to index *n_steps_done.  f_var_last [N][3] nullable: f_var of
 * the last sample.
 * ------------------------------------------------------------------------------------------ */
int oracle_md_switching(const oracle_hparams *hp, const oracle_weights *w, int64_t N, double *x, double *v,
                        const double *masses, const int32_t *species, const double *L, const int32_t *pbc,
                        double skin, double dt, int64_t n_steps, int64_t sampling_rate, double f_sigma_stop,
                        double *epot, double *ekin, double *sigma_e, double *sigma_f_max, double *f_var_last,
                        int64_t *n_steps_done, int64_t *n_samples, int64_t *n_rebuilds) {
    if (sampling_rate < 1 || hp->n_heads > 64) return -1;
    const int M = hp->n_heads;
    pairlist_t pl = {0, 0, NULL, NULL, NULL};
    double *F = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    double *Eh = (double *)malloc(sizeof(double) * (size_t)N * M);
    double *xu = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    double *xref = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    double *em = (double *)malloc(sizeof(double) * (size_t)N), *ev = (double *)malloc(sizeof(double) * (size_t)N);
    double *fm = (double *)malloc(sizeof(double) * 3 * (size_t)N), *fv = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    double hw[64];
    for (int m = 0; m < M; ++m) hw[m] = 1.0 / M;
    int64_t rebuilds = 0, samples = 0, done = 0;
    for (int64_t i = 0; i < N; ++i) wrap_position(x + 3 * i, L, pbc);
    memcpy(xu, x, sizeof(double) * 3 * (size_t)N);
    memcpy(xref, x, sizeof(double) * 3 * (size_t)N);
    build_list(&pl, N, x, L, pbc, hp->r_cut + skin);
    oracle_energy_forces(hp, w, N, xu, species, L, pl.n, pl.i, pl.j, pl.n3, hw, Eh, F, NULL, NULL, NULL, NULL, NULL);
    for (int64_t step = 0;; ++step) {
        double ep = 0.0, ek = 0.0;
        for (int64_t i = 0; i < N; ++i) {
            for (int m = 0; m < M; ++m) ep += hw[m] * Eh[(size_t)i * M + m];
            ek += 0.5 * masses[i] * (v[3 * i] * v[3 * i] + v[3 * i + 1] * v[3 * i + 1] + v[3 * i + 2] * v[3 * i + 2]);
        }
        epot[step] = ep;
        ekin[step] = ek / ACC_CONV;
        done = step;
        if (step > 0 && step % sampling_rate == 0) {
            oracle_ensemble(hp, w, N, xu, species, L, pl.n, pl.i, pl.j, pl.n3, Eh, em, ev, fm, fv, NULL);
            double tot[64], mean = 0.0, var = 0.0, worst = 0.0;
            for (int m = 0; m < M; ++m) {
                tot[m] = 0.0;
                for (int64_t i = 0; i < N; ++i) tot[m] += Eh[(size_t)i * M + m];
                mean += tot[m];
            }
            mean /= M;
            for (int m = 0; m < M; ++m) var += (tot[m] - mean) * (tot[m] - mean);
            for (int64_t i = 0; i < N; ++i) {
                const double sf = sqrt(fv[3 * i] + fv[3 * i + 1] + fv[3 * i + 2]);
                if (sf > worst) worst = sf;
            }
            sigma_e[samples] = sqrt(var / M);
            sigma_f_max[samples] = worst;
            ++samples;
            if (f_var_last) memcpy(f_var_last, fv, sizeof(double) * 3 * (size_t)N);
            if (f_sigma_stop > 0.0 && worst > f_sigma_stop) break;
        }
        if (step == n_steps) break;
        double maxd2 = 0.0;
        for (int64_t i = 0; i < N; ++i) {
            double d2 = 0.0;
            for (int a = 0; a < 3; ++a) {
                v[3 * i + a] += 0.5 * dt * F[3 * i + a] / masses[i] * ACC_CONV;
                xu[3 * i + a] += dt * v[3 * i + a];
                x[3 * i + a] = xu[3 * i + a];
                double dd = xu[3 * i + a] - xref[3 * i + a];
                d2 += dd * dd;
            }
            wrap_position(x + 3 * i, L, pbc);
            if (d2 > maxd2) maxd2 = d2;
        }
        if (sqrt(maxd2) > 0.5 * skin) {
            memcpy(xu, x, sizeof(double) * 3 * (size_t)N);
            memcpy(xref, x, sizeof(double) * 3 * (size_t)N);
            build_list(&pl, N, x, L, pbc, hp->r_cut + skin);
            ++rebuilds;
        }
        oracle_energy_forces(hp, w, N, xu, species, L, pl.n, pl.i, pl.j, pl.n3, hw, Eh, F, NULL, NULL, NULL, NULL, NULL);
        for (int64_t i = 0; i < N; ++i)
            for (int a = 0; a < 3; ++a) v[3 * i + a] += 0.5 * dt * F[3 * i + a] / masses[i] * ACC_CONV;
    }
    if (n_steps_done) *n_steps_done = done;
    if (n_samples) *n_samples = samples;
    if (n_rebuilds) *n_rebuilds = rebuilds;
    free(F); free(Eh); free(xu); free(xref); free(em); free(ev); free(fm); free(fv);
    free(pl.i); free(pl.j); free(pl.n3);
    return 0;
}
