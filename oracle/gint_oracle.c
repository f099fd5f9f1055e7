/*
 * gint_oracle.c — CPU ORACLE for real-space grid integration (TEST INFRASTRUCTURE ONLY).
 *
 * This file is the plain, slow, double-precision definition of what the GPU path
 * computes.  It is test infrastructure: only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with paper_2409_09399_b200/csrc (the CUDA path).
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md):
 *   Eq. 2  H_{mu nu} = sum_r phi_mu(r-R_mu) V(r) phi_nu(r-R_nu) dV
 *   Eq. 3  rho(r)    = sum_{mu nu} rho_{mu nu} phi_mu(r-R_mu) phi_nu(r-R_nu)
 *   neighbour rule: an atom contributes at a grid point iff the
 *   distance is LESS than its cutoff radius; otherwise its orbitals are zero there
 *   (Fig. 6).
 * The paper is silent on the orbital convention, the radial interpolation, the mesh
 * indexing and periodic images; the readings used here are DESIGN.md "Readings"
 * R1..R9.
 *
 * Parity pins (tests/test_oracle_pins.py): H symmetry, V==1 -> overlap with closed-form
 * on-site values, sum rho dV = Tr(D S), sum V rho dV = <D,H>, closed-form Gaussian
 * overlap, brute force on 1-2 atoms, translation / permutation invariance.
 * Individual H or rho values of the paper's own systems: PARITY UNPINNED (the paper
 * prints none).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_MAX_L 2
#define ORACLE_MAX_ORB 64

typedef struct {
    int n_species;
    const int *n_shell;     /* [n_species] */
    const int *shell_l;     /* concatenated */
    const double *rcut;     /* [n_species] */
    double dr;
    const int *n_knot;      /* [n_species] knots per shell */
    const double *tab_y;    /* concatenated [species][shell][knot] */
    const double *tab_y2;
    /* derived */
    int *shell_off;         /* [n_species] first shell index of species */
    long long *tab_off;     /* [total shells] offset of each shell table */
    int *norb;              /* [n_species] */
} basis_t;

static int basis_setup(basis_t *b) {
    int ns = b->n_species, tot = 0;
    b->shell_off = (int *)malloc(sizeof(int) * (ns + 1));
    b->norb = (int *)malloc(sizeof(int) * ns);
    for (int s = 0; s < ns; s++) { b->shell_off[s] = tot; tot += b->n_shell[s]; }
    b->shell_off[ns] = tot;
    b->tab_off = (long long *)malloc(sizeof(long long) * (tot + 1));
    long long off = 0;
    for (int s = 0; s < ns; s++) {
        int no = 0;
        for (int k = b->shell_off[s]; k < b->shell_off[s + 1]; k++) {
            if (b->shell_l[k] < 0 || b->shell_l[k] > ORACLE_MAX_L) return -1;
            b->tab_off[k] = off; off += b->n_knot[s];
            no += 2 * b->shell_l[k] + 1;
        }
        if (no > ORACLE_MAX_ORB) return -1;
        b->norb[s] = no;
    }
    b->tab_off[tot] = off;
    return 0;
}
static void basis_free(basis_t *b) { free(b->shell_off); free(b->tab_off); free(b->norb); }

/* R5: cubic spline on knots r_i = i*dr:
 *   i = min(floor(r/dr), n-1), b = r/dr - i, a = 1-b,
 *   R = a*y_i + b*y_{i+1} + [(a^3-a)*y''_i + (b^3-b)*y''_{i+1}] * dr^2/6          */
static double radial(const basis_t *bs, int species, int shell, double r) {
    int n = bs->n_knot[species] - 1;               /* intervals */
    const double *y  = bs->tab_y  + bs->tab_off[bs->shell_off[species] + shell];
    const double *y2 = bs->tab_y2 + bs->tab_off[bs->shell_off[species] + shell];
    double x = r / bs->dr;
    int i = (int)floor(x);
    if (i > n - 1) i = n - 1;
    if (i < 0) i = 0;
    double b = x - (double)i, a = 1.0 - b;
    return a * y[i] + b * y[i + 1]
         + ((a * a * a - a) * y2[i] + (b * b * b - b) * y2[i + 1]) * (bs->dr * bs->dr) / 6.0;
}

/* R3/R4: phi_{A,s,m}(d) = R_s(|d|) * Y_{l_s m}(d/|d|), zero when |d| >= rc.
 * Real spherical harmonics, m = -l..l, no Condon-Shortley phase:
 *   l=0: 1/(2 sqrt(pi))
 *   l=1: sqrt(3/4pi) * (y, z, x)
 *   l=2: sqrt(15/4pi)*xy, sqrt(15/4pi)*yz, sqrt(5/16pi)*(3z^2-1), sqrt(15/4pi)*xz, sqrt(15/16pi)*(x^2-y^2)
 * At |d| < 1e-12 only l=0 orbitals are non-zero.  Returns 1 if inside the sphere. */
static int phi_eval(const basis_t *bs, int species, const double d[3], double *out) {
    const double PI = 3.14159265358979323846;
    int no = bs->norb[species];
    double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    if (!(r < bs->rcut[species])) { for (int k = 0; k < no; k++) out[k] = 0.0; return 0; }
    double x = 0, y = 0, z = 0; int tiny = (r < 1e-12);
    if (!tiny) { x = d[0] / r; y = d[1] / r; z = d[2] / r; }
    int o = 0, nsh = bs->n_shell[species];
    for (int s = 0; s < nsh; s++) {
        int l = bs->shell_l[bs->shell_off[species] + s];
        double R = radial(bs, species, s, r);
        if (l == 0) {
            out[o++] = R * (0.5 / sqrt(PI));
        } else if (l == 1) {
            double c = sqrt(3.0 / (4.0 * PI));
            if (tiny) { out[o++] = 0; out[o++] = 0; out[o++] = 0; }
            else { out[o++] = R * c * y; out[o++] = R * c * z; out[o++] = R * c * x; }
        } else {
            double c = sqrt(15.0 / (4.0 * PI));
            if (tiny) { for (int k = 0; k < 5; k++) out[o++] = 0; }
            else {
                out[o++] = R * c * x * y;
                out[o++] = R * c * y * z;
                out[o++] = R * sqrt(5.0 / (16.0 * PI)) * (3.0 * z * z - 1.0);
                out[o++] = R * c * x * z;
                out[o++] = R * 0.5 * c * (x * x - y * y);
            }
        }
    }
    return 1;
}

/* ---- geometry helpers ------------------------------------------------------------ */
static double det3(const double c[9]) {
    return c[0] * (c[4] * c[8] - c[5] * c[7]) - c[1] * (c[3] * c[8] - c[5] * c[6]) + c[2] * (c[3] * c[7] - c[4] * c[6]);
}
static void inv3(const double c[9], double inv[9]) {   /* inv such that frac = pos * inv  (row vectors) */
    double d = det3(c);
    inv[0] = (c[4] * c[8] - c[5] * c[7]) / d; inv[1] = (c[2] * c[7] - c[1] * c[8]) / d; inv[2] = (c[1] * c[5] - c[2] * c[4]) / d;
    inv[3] = (c[5] * c[6] - c[3] * c[8]) / d; inv[4] = (c[0] * c[8] - c[2] * c[6]) / d; inv[5] = (c[2] * c[3] - c[0] * c[5]) / d;
    inv[6] = (c[3] * c[7] - c[4] * c[6]) / d; inv[7] = (c[1] * c[6] - c[0] * c[7]) / d; inv[8] = (c[0] * c[4] - c[1] * c[3]) / d;
}
/* height of the cell along direction i = 1/|column i of inv| (distance between the lattice planes) */
static void heights(const double inv[9], double h[3]) {
    for (int i = 0; i < 3; i++) h[i] = 1.0 / sqrt(inv[i] * inv[i] + inv[3 + i] * inv[3 + i] + inv[6 + i] * inv[6 + i]);
}
static void to_frac(const double inv[9], const double p[3], double f[3]) {
    for (int i = 0; i < 3; i++) f[i] = p[0] * inv[i] + p[1] * inv[3 + i] + p[2] * inv[6 + i];
}
static void lattice(const double cell[9], int n1, int n2, int n3, double R[3]) {
    for (int k = 0; k < 3; k++) R[k] = n1 * cell[k] + n2 * cell[3 + k] + n3 * cell[6 + k];
}

/* ---- R7: pair keys ---------------------------------------------------------------
 * All ordered keys p = (A, B, n) with |tau_B + R_n - tau_A| < rc_A + rc_B (strict), incl.
 * (A,A,0) and (A,A,n!=0); order lexicographic in (A, B, n1, n2, n3); block p is row-major
 * norb(A) x norb(B) at offset[p].  Two-pass: call with pA==NULL to count.               */
long long oracle_pairs(int n_species, const int *n_shell, const int *shell_l, const double *rcut,
                       int n_atoms, const int *atom_species, const double *atom_pos, const double cell[9],
                       int *pA, int *pB, int *pR, long long *offset)
{
    double inv[9], h[3];
    if (!(det3(cell) > 0)) return -1;
    inv3(cell, inv); heights(inv, h);
    int *norb = (int *)malloc(sizeof(int) * n_species);
    for (int s = 0, k = 0; s < n_species; s++) { norb[s] = 0; for (int q = 0; q < n_shell[s]; q++, k++) norb[s] += 2 * shell_l[k] + 1; }
    long long np = 0, off = 0;
    for (int A = 0; A < n_atoms; A++) {
        for (int B = 0; B < n_atoms; B++) {
            double rmax = rcut[atom_species[A]] + rcut[atom_species[B]];
            double dcart[3] = { atom_pos[3 * B] - atom_pos[3 * A], atom_pos[3 * B + 1] - atom_pos[3 * A + 1], atom_pos[3 * B + 2] - atom_pos[3 * A + 2] };
            double f[3]; to_frac(inv, dcart, f);
            int lo[3], hi[3];
            for (int i = 0; i < 3; i++) { lo[i] = (int)floor(-f[i] - rmax / h[i]) - 1; hi[i] = (int)ceil(-f[i] + rmax / h[i]) + 1; }
            for (int n1 = lo[0]; n1 <= hi[0]; n1++)
            for (int n2 = lo[1]; n2 <= hi[1]; n2++)
            for (int n3 = lo[2]; n3 <= hi[2]; n3++) {
                double R[3]; lattice(cell, n1, n2, n3, R);
                double dx = dcart[0] + R[0], dy = dcart[1] + R[1], dz = dcart[2] + R[2];
                if (sqrt(dx * dx + dy * dy + dz * dz) < rmax) {
                    if (pA) { pA[np] = A; pB[np] = B; pR[3 * np] = n1; pR[3 * np + 1] = n2; pR[3 * np + 2] = n3; offset[np] = off; }
                    np++; off += (long long)norb[atom_species[A]] * norb[atom_species[B]];
                }
            }
        }
    }
    if (pA) offset[np] = off;
    free(norb);
    return np;
}

/* single-point orbital evaluation, exported for the pins */
int oracle_phi(int n_species, const int *n_shell, const int *shell_l, const double *rcut, double dr,
               const int *n_knot, const double *tab_y, const double *tab_y2,
               int species, const double d[3], double *out)
{
    basis_t bs = { n_species, n_shell, shell_l, rcut, dr, n_knot, tab_y, tab_y2, 0, 0, 0 };
    if (basis_setup(&bs)) return -1;
    int in = phi_eval(&bs, species, d, out);
    basis_free(&bs);
    return in;
}

int oracle_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static long long imod(long long a, long long n) { long long r = a % n; return r < 0 ? r + n : r; }

/* ---- R8 / Eq. 2: H blocks, pair-major direct loops --------------------------------
 * H_p[mu,nu] = dV * sum over ALL-SPACE mesh points r of V(r) phi_{A mu}(r - tau_A) phi_{B nu}(r - tau_B - R_n)
 * (V periodic: index wrapped into the home mesh).  Mesh: r = (i/N1) a1 + (j/N2) a2 + (k/N3) a3,
 * g = (i*N2 + j)*N3 + k, dV = det(cell)/(N1 N2 N3)  (R1).  Only mesh points inside the
 * fractional bounding box of sphere A are visited; points outside either sphere add zero.
 * sel == NULL: all pairs; else only pair indices sel[0..n_sel) are computed (others untouched). */
int oracle_vlocal(int n_species, const int *n_shell, const int *shell_l, const double *rcut, double dr,
                  const int *n_knot, const double *tab_y, const double *tab_y2,
                  int n_atoms, const int *atom_species, const double *atom_pos, const double cell[9], const int mesh[3],
                  const double *V, long long n_pairs, const int *pA, const int *pB, const int *pR, const long long *offset,
                  double *H, long long n_sel, const long long *sel)
{
    basis_t bs = { n_species, n_shell, shell_l, rcut, dr, n_knot, tab_y, tab_y2, 0, 0, 0 };
    if (basis_setup(&bs)) return -1;
    double inv[9], h[3]; inv3(cell, inv); heights(inv, h);
    const int N1 = mesh[0], N2 = mesh[1], N3 = mesh[2];
    const double dV = det3(cell) / ((double)N1 * N2 * N3);
    long long ntask = sel ? n_sel : n_pairs;
    (void)n_atoms;
#pragma omp parallel for schedule(dynamic, 1)
    for (long long q = 0; q < ntask; q++) {
        long long p = sel ? sel[q] : q;
        int A = pA[p], B = pB[p], sA = atom_species[A], sB = atom_species[B];
        int nA = bs.norb[sA], nB = bs.norb[sB];
        double acc[ORACLE_MAX_ORB * ORACLE_MAX_ORB];
        for (int k = 0; k < nA * nB; k++) acc[k] = 0.0;
        const double *tA = atom_pos + 3 * A;
        double R[3]; lattice(cell, pR[3 * p], pR[3 * p + 1], pR[3 * p + 2], R);
        double tB[3] = { atom_pos[3 * B] + R[0], atom_pos[3 * B + 1] + R[1], atom_pos[3 * B + 2] + R[2] };
        double fA[3]; to_frac(inv, tA, fA);
        double rcA = rcut[sA];
        long long lo[3], hi[3]; const int NN[3] = { N1, N2, N3 };
        for (int i = 0; i < 3; i++) {
            lo[i] = (long long)floor((fA[i] - rcA / h[i]) * NN[i]) - 1;
            hi[i] = (long long)ceil((fA[i] + rcA / h[i]) * NN[i]) + 1;
        }
        double pa[ORACLE_MAX_ORB], pb[ORACLE_MAX_ORB];
        for (long long i = lo[0]; i <= hi[0]; i++)
        for (long long j = lo[1]; j <= hi[1]; j++)
        for (long long k = lo[2]; k <= hi[2]; k++) {
            double u = (double)i / N1, v = (double)j / N2, w = (double)k / N3;
            double r[3] = { u * cell[0] + v * cell[3] + w * cell[6], u * cell[1] + v * cell[4] + w * cell[7], u * cell[2] + v * cell[5] + w * cell[8] };
            double dA[3] = { r[0] - tA[0], r[1] - tA[1], r[2] - tA[2] };
            if (!phi_eval(&bs, sA, dA, pa)) continue;
            double dB[3] = { r[0] - tB[0], r[1] - tB[1], r[2] - tB[2] };
            if (!phi_eval(&bs, sB, dB, pb)) continue;
            double Vg = V[(imod(i, N1) * N2 + imod(j, N2)) * N3 + imod(k, N3)];
            for (int mu = 0; mu < nA; mu++) {
                double t = Vg * pa[mu];
                for (int nu = 0; nu < nB; nu++) acc[mu * nB + nu] += t * pb[nu];
            }
        }
        double *Hp = H + offset[p];
        for (int k = 0; k < nA * nB; k++) Hp[k] = acc[k] * dV;
    }
    basis_free(&bs);
    return 0;
}

/* ---- R9 / Eq. 3: density, point-major direct loops ----------------------------------
 * rho_g = sum over ORDERED pairs of atom images ((A,t),(B,t')) non-zero at r_g of
 *         phi_A(r_g;t)^T  D_(A,B,t'-t)  phi_B(r_g;t')          (no symmetry of D assumed).
 * Images are found by scanning a coarse bin list (own code, conservative), then the strict
 * |d| < rc test inside phi_eval decides.  Block lookup: binary search in the sorted key list.
 * sel == NULL: all mesh points; else only mesh indices sel[0..n_sel) are written.
 * Returns 0, or -2 if a needed key is missing from the pair list.                          */
typedef struct { int A; int t[3]; double pos[3]; } image_t;

static long long find_pair(const long long *row, const int *pB, const int *pR, int A, int B, const int n[3]) {
    long long lo = row[A], hi = row[A + 1] - 1;
    while (lo <= hi) {
        long long m = (lo + hi) / 2; int c;
        if (pB[m] != B) c = pB[m] < B ? -1 : 1;
        else if (pR[3 * m] != n[0]) c = pR[3 * m] < n[0] ? -1 : 1;
        else if (pR[3 * m + 1] != n[1]) c = pR[3 * m + 1] < n[1] ? -1 : 1;
        else if (pR[3 * m + 2] != n[2]) c = pR[3 * m + 2] < n[2] ? -1 : 1;
        else return m;
        if (c < 0) lo = m + 1; else hi = m - 1;
    }
    return -1;
}

int oracle_rho(int n_species, const int *n_shell, const int *shell_l, const double *rcut, double dr,
               const int *n_knot, const double *tab_y, const double *tab_y2,
               int n_atoms, const int *atom_species, const double *atom_pos, const double cell[9], const int mesh[3],
               const double *D, long long n_pairs, const int *pA, const int *pB, const int *pR, const long long *offset,
               double *rho, long long n_sel, const long long *sel)
{
    basis_t bs = { n_species, n_shell, shell_l, rcut, dr, n_knot, tab_y, tab_y2, 0, 0, 0 };
    if (basis_setup(&bs)) return -1;
    double inv[9], h[3]; inv3(cell, inv); heights(inv, h);
    const int N1 = mesh[0], N2 = mesh[1], N3 = mesh[2];

    /* row starts of the sorted key list */
    long long *row = (long long *)malloc(sizeof(long long) * (n_atoms + 1));
    { long long p = 0; for (int A = 0; A <= n_atoms; A++) { while (p < n_pairs && pA[p] < A) p++; row[A] = p; } }

    /* all images whose sphere can reach the home cell: frac coords in (-rho_i, 1+rho_i) */
    long long n_img = 0, cap = 1024; image_t *img = (image_t *)malloc(sizeof(image_t) * cap);
    for (int A = 0; A < n_atoms; A++) {
        double f[3]; to_frac(inv, atom_pos + 3 * A, f);
        double rc = rcut[atom_species[A]]; int lo[3], hi[3];
        for (int i = 0; i < 3; i++) { lo[i] = (int)floor(-f[i] - rc / h[i]) - 1; hi[i] = (int)ceil(1.0 - f[i] + rc / h[i]) + 1; }
        for (int t1 = lo[0]; t1 <= hi[0]; t1++) for (int t2 = lo[1]; t2 <= hi[1]; t2++) for (int t3 = lo[2]; t3 <= hi[2]; t3++) {
            double g[3] = { f[0] + t1, f[1] + t2, f[2] + t3 }; int ok = 1;
            for (int i = 0; i < 3; i++) if (g[i] + rc / h[i] < 0.0 || g[i] - rc / h[i] > 1.0) ok = 0;
            if (!ok) continue;
            if (n_img == cap) { cap *= 2; img = (image_t *)realloc(img, sizeof(image_t) * cap); }
            double R[3]; lattice(cell, t1, t2, t3, R);
            image_t *q = &img[n_img++]; q->A = A; q->t[0] = t1; q->t[1] = t2; q->t[2] = t3;
            for (int k = 0; k < 3; k++) q->pos[k] = atom_pos[3 * A + k] + R[k];
        }
    }
    /* coarse bins over the home cell in fractional coordinates (bin width >= ~2 bohr);
     * an image is listed in every bin its fractional bounding box touches (conservative) */
    int nb[3];
    for (int i = 0; i < 3; i++) { nb[i] = (int)floor(h[i] / 2.0); if (nb[i] < 1) nb[i] = 1; if (nb[i] > 128) nb[i] = 128; }
    long long nbin = (long long)nb[0] * nb[1] * nb[2];
    long long *bstart = (long long *)calloc(nbin + 1, sizeof(long long));
    long long *fill = (long long *)calloc(nbin, sizeof(long long));
    int *blist = 0;
    for (int pass = 0; pass < 2; pass++) {
        for (long long q = 0; q < n_img; q++) {
            double f[3]; to_frac(inv, img[q].pos, f); double rc = rcut[atom_species[img[q].A]];
            int lo[3], hi[3];
            for (int i = 0; i < 3; i++) {
                lo[i] = (int)floor((f[i] - rc / h[i]) * nb[i]) - 1; if (lo[i] < 0) lo[i] = 0;
                hi[i] = (int)floor((f[i] + rc / h[i]) * nb[i]) + 1; if (hi[i] > nb[i] - 1) hi[i] = nb[i] - 1;
            }
            for (int b1 = lo[0]; b1 <= hi[0]; b1++) for (int b2 = lo[1]; b2 <= hi[1]; b2++) for (int b3 = lo[2]; b3 <= hi[2]; b3++) {
                long long b = ((long long)b1 * nb[1] + b2) * nb[2] + b3;
                if (pass == 0) bstart[b + 1]++; else blist[bstart[b] + fill[b]++] = (int)q;
            }
        }
        if (pass == 0) {
            for (long long b = 0; b < nbin; b++) bstart[b + 1] += bstart[b];
            blist = (int *)malloc(sizeof(int) * (bstart[nbin] > 0 ? bstart[nbin] : 1));
        }
    }

    long long npts = sel ? n_sel : (long long)N1 * N2 * N3;
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(| : bad)
    for (long long s = 0; s < npts; s++) {
        long long g = sel ? sel[s] : s;
        long long k = g % N3, j = (g / N3) % N2, i = g / ((long long)N3 * N2);
        double u = (double)i / N1, v = (double)j / N2, w = (double)k / N3;
        double r[3] = { u * cell[0] + v * cell[3] + w * cell[6], u * cell[1] + v * cell[4] + w * cell[7], u * cell[2] + v * cell[5] + w * cell[8] };
        int b1 = (int)(u * nb[0]), b2 = (int)(v * nb[1]), b3 = (int)(w * nb[2]);
        if (b1 > nb[0] - 1) b1 = nb[0] - 1;
        if (b2 > nb[1] - 1) b2 = nb[1] - 1;
        if (b3 > nb[2] - 1) b3 = nb[2] - 1;
        long long b = ((long long)b1 * nb[1] + b2) * nb[2] + b3;
        /* list of images non-zero at r_g, with their orbital vectors */
        int cnt = 0, capl = 64; int *who = (int *)malloc(sizeof(int) * capl);
        double *val = (double *)malloc(sizeof(double) * capl * ORACLE_MAX_ORB);
        for (long long c = bstart[b]; c < bstart[b + 1]; c++) {
            const image_t *im = &img[blist[c]];
            double d[3] = { r[0] - im->pos[0], r[1] - im->pos[1], r[2] - im->pos[2] };
            if (cnt == capl) { capl *= 2; who = (int *)realloc(who, sizeof(int) * capl); val = (double *)realloc(val, sizeof(double) * capl * ORACLE_MAX_ORB); }
            if (phi_eval(&bs, atom_species[im->A], d, val + (size_t)cnt * ORACLE_MAX_ORB)) who[cnt++] = blist[c];
        }
        double sum = 0.0;
        for (int a = 0; a < cnt; a++) for (int c = 0; c < cnt; c++) {
            const image_t *ia = &img[who[a]], *ib = &img[who[c]];
            int n[3] = { ib->t[0] - ia->t[0], ib->t[1] - ia->t[1], ib->t[2] - ia->t[2] };
            long long p = find_pair(row, pB, pR, ia->A, ib->A, n);
            if (p < 0) { bad |= 1; continue; }
            int nA = bs.norb[atom_species[ia->A]], nB = bs.norb[atom_species[ib->A]];
            const double *Dp = D + offset[p];
            const double *pa = val + (size_t)a * ORACLE_MAX_ORB, *pb = val + (size_t)c * ORACLE_MAX_ORB;
            for (int mu = 0; mu < nA; mu++) {
                double t = 0.0;
                for (int nu = 0; nu < nB; nu++) t += Dp[mu * nB + nu] * pb[nu];
                sum += pa[mu] * t;
            }
        }
        rho[g] = sum;
        free(who); free(val);
    }
    free(bstart); free(blist); free(fill); free(img); free(row); basis_free(&bs);
    return bad ? -2 : 0;
}

/* =====================================================================================
 * Pulay force and stress of the local-potential energy (Eq. 4 and Eq. 5; orbital gradients PAPER.md:163).
 *
 * Reading R15: with E = sum_keys <D_key, H_key> = dV sum_g V_g rho_g (identity P4), at FIXED V (values per mesh index),
 * D and dV,
 *   F_C^a      = - dE / d tau_C^a
 *              = dV sum_{r in all space} V(r) sum_i  d_a phi_{C i}(r - tau_C)  Psi_{C i}(r),
 *   Psi_{C i}(r) = sum_{keys (C,B,n)} sum_j ( D_(C,B,n)[i][j] + D_(B,C,-n)[j][i] ) phi_{B j}(r - tau_B - R_n)
 * (moving atom C changes phi_C in every key it heads and, through the mirror key, every key it ends; d phi(r - tau)/d tau = - grad phi),
 *   sigma^{ab} = - (1/Omega) dE / d eps_ab   under r -> (1 + eps) r of atoms AND mesh points
 *              = - (1/Omega) sum_C dV sum_r V(r) sum_i d_a phi_{C i} Psi_{C i} (r - tau_C)^b .
 * Eq. 4 prints a factor 1/Omega for the force as well: dropped (a force is an energy derivative, the factor belongs to Eq. 5);
 * Eq. 5 prints tau^b: read as the position of the atom relative to the integration point (the only translation-invariant reading).
 *
 * Orbital gradient: phi = R(r) Y(u), u = d / r, Y = c P_l(u) with P_l a homogeneous polynomial of degree l
 * (3 z^2 - 1 == 2 z^2 - x^2 - y^2 on the unit sphere):
 *   grad phi = (R' - l R / r) u Y + (R / r) c grad_u P_l(u),
 *   R'(r) = [ (y_{i+1} - y_i) - (3 a^2 - 1) y''_i dr^2/6 + (3 b^2 - 1) y''_{i+1} dr^2/6 ] / dr   (derivative of the spline of R5).
 * At |d| < 1e-12 the direction is undefined: grad phi = 0 for l = 0 and l = 2, and c_1 R'(0) e_m for l = 1 (the limit of R / r).
 * Pins (tests/test_oracle_pins.py): central finite differences of E through oracle_vlocal (atoms displaced; cell strained),
 * an independent brute force with scipy's spline derivative on a skew two-species cell, sum of forces under a rigid shift.
 * sel == NULL: all atoms, sigma is written; else only the forces of atoms sel[0..n_sel) are written and sigma is left alone. */
static double radial_d1(const basis_t *bs, int species, int shell, double r) {
    int n = bs->n_knot[species] - 1;
    const double *y  = bs->tab_y  + bs->tab_off[bs->shell_off[species] + shell];
    const double *y2 = bs->tab_y2 + bs->tab_off[bs->shell_off[species] + shell];
    double x = r / bs->dr;
    int i = (int)floor(x);
    if (i > n - 1) i = n - 1;
    if (i < 0) i = 0;
    double b = x - (double)i, a = 1.0 - b;
    return (y[i + 1] - y[i]) / bs->dr
         + (-(3.0 * a * a - 1.0) * y2[i] + (3.0 * b * b - 1.0) * y2[i + 1]) * bs->dr / 6.0;
}

/* values out[norb] and gradients grad[norb][3]; returns 1 if inside the sphere */
static int dphi_eval(const basis_t *bs, int species, const double d[3], double *out, double *grad) {
    const double PI = 3.14159265358979323846;
    int no = bs->norb[species];
    double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    if (!(r < bs->rcut[species])) { for (int k = 0; k < no; k++) { out[k] = 0.0; grad[3 * k] = grad[3 * k + 1] = grad[3 * k + 2] = 0.0; } return 0; }
    phi_eval(bs, species, d, out);
    int tiny = (r < 1e-12);
    double u[3] = { 0, 0, 0 };
    if (!tiny) { u[0] = d[0] / r; u[1] = d[1] / r; u[2] = d[2] / r; }
    double x = u[0], y = u[1], z = u[2];
    int o = 0, nsh = bs->n_shell[species];
    for (int s = 0; s < nsh; s++) {
        int l = bs->shell_l[bs->shell_off[species] + s];
        double R = radial(bs, species, s, r), R1 = radial_d1(bs, species, s, r);
        int nm = 2 * l + 1;
        double c[5], P[5], gP[5][3];
        if (l == 0) {
            c[0] = 0.5 / sqrt(PI); P[0] = 1.0; gP[0][0] = gP[0][1] = gP[0][2] = 0.0;
        } else if (l == 1) {
            double c1 = sqrt(3.0 / (4.0 * PI));
            for (int m = 0; m < 3; m++) { c[m] = c1; gP[m][0] = gP[m][1] = gP[m][2] = 0.0; }
            P[0] = y; gP[0][1] = 1.0;  P[1] = z; gP[1][2] = 1.0;  P[2] = x; gP[2][0] = 1.0;
        } else {
            double c2 = sqrt(15.0 / (4.0 * PI));
            c[0] = c2; P[0] = x * y;  gP[0][0] = y; gP[0][1] = x; gP[0][2] = 0.0;
            c[1] = c2; P[1] = y * z;  gP[1][0] = 0.0; gP[1][1] = z; gP[1][2] = y;
            c[2] = sqrt(5.0 / (16.0 * PI)); P[2] = 2.0 * z * z - x * x - y * y; gP[2][0] = -2.0 * x; gP[2][1] = -2.0 * y; gP[2][2] = 4.0 * z;
            c[3] = c2; P[3] = x * z;  gP[3][0] = z; gP[3][1] = 0.0; gP[3][2] = x;
            c[4] = 0.5 * c2; P[4] = x * x - y * y; gP[4][0] = 2.0 * x; gP[4][1] = -2.0 * y; gP[4][2] = 0.0;
        }
        for (int m = 0; m < nm; m++, o++) {
            for (int a = 0; a < 3; a++) {
                if (tiny) grad[3 * o + a] = (l == 1) ? c[m] * R1 * gP[m][a] : 0.0;
                else grad[3 * o + a] = (R1 - l * R / r) * u[a] * c[m] * P[m] + (R / r) * c[m] * gP[m][a];
            }
        }
    }
    return 1;
}

/* single-point orbital gradient, exported for the pins */
int oracle_dphi(int n_species, const int *n_shell, const int *shell_l, const double *rcut, double dr,
                const int *n_knot, const double *tab_y, const double *tab_y2,
                int species, const double d[3], double *out, double *grad)
{
    basis_t bs = { n_species, n_shell, shell_l, rcut, dr, n_knot, tab_y, tab_y2, 0, 0, 0 };
    if (basis_setup(&bs)) return -1;
    int in = dphi_eval(&bs, species, d, out, grad);
    basis_free(&bs);
    return in;
}

int oracle_force_stress(int n_species, const int *n_shell, const int *shell_l, const double *rcut, double dr,
                        const int *n_knot, const double *tab_y, const double *tab_y2,
                        int n_atoms, const int *atom_species, const double *atom_pos, const double cell[9], const int mesh[3],
                        const double *V, const double *D, long long n_pairs, const int *pA, const int *pB, const int *pR, const long long *offset,
                        double *F, double *sigma, long long n_sel, const long long *sel)
{
    basis_t bs = { n_species, n_shell, shell_l, rcut, dr, n_knot, tab_y, tab_y2, 0, 0, 0 };
    if (basis_setup(&bs)) return -1;
    double inv[9], h[3]; inv3(cell, inv); heights(inv, h);
    const int N1 = mesh[0], N2 = mesh[1], N3 = mesh[2];
    const double Omega = det3(cell), dV = Omega / ((double)N1 * N2 * N3);
    long long *row = (long long *)malloc(sizeof(long long) * (n_atoms + 1));
    { long long p = 0; for (int A = 0; A <= n_atoms; A++) { while (p < n_pairs && pA[p] < A) p++; row[A] = p; } }
    long long ntask = sel ? n_sel : n_atoms;
    double sg[9] = { 0, 0, 0, 0, 0, 0, 0, 0, 0 };
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(| : bad) reduction(+ : sg[:9])
    for (long long q = 0; q < ntask; q++) {
        int C = sel ? (int)sel[q] : (int)q, sC = atom_species[C], nC = bs.norb[sC];
        const double *tC = atom_pos + 3 * C;
        double fC[3]; to_frac(inv, tC, fC);
        double rcC = rcut[sC];
        long long lo[3], hi[3]; const int NN[3] = { N1, N2, N3 };
        for (int i = 0; i < 3; i++) {
            lo[i] = (long long)floor((fC[i] - rcC / h[i]) * NN[i]) - 1;
            hi[i] = (long long)ceil((fC[i] + rcC / h[i]) * NN[i]) + 1;
        }
        /* mirror key (B, C, -n) of every key (C, B, n) of row C */
        long long nk = row[C + 1] - row[C];
        long long *mir = (long long *)malloc(sizeof(long long) * (nk > 0 ? nk : 1));
        for (long long k = 0; k < nk; k++) {
            long long p = row[C] + k; int mn[3] = { -pR[3 * p], -pR[3 * p + 1], -pR[3 * p + 2] };
            mir[k] = find_pair(row, pB, pR, pB[p], C, mn);
            if (mir[k] < 0) bad |= 1;
        }
        double Fc[3] = { 0, 0, 0 };
        double pc[ORACLE_MAX_ORB], gc[3 * ORACLE_MAX_ORB], pb[ORACLE_MAX_ORB], psi[ORACLE_MAX_ORB];
        for (long long i = lo[0]; i <= hi[0] && !bad; i++)
        for (long long j = lo[1]; j <= hi[1]; j++)
        for (long long k = lo[2]; k <= hi[2]; k++) {
            double u = (double)i / N1, v = (double)j / N2, w = (double)k / N3;
            double r[3] = { u * cell[0] + v * cell[3] + w * cell[6], u * cell[1] + v * cell[4] + w * cell[7], u * cell[2] + v * cell[5] + w * cell[8] };
            double dC[3] = { r[0] - tC[0], r[1] - tC[1], r[2] - tC[2] };
            if (!dphi_eval(&bs, sC, dC, pc, gc)) continue;
            for (int m = 0; m < nC; m++) psi[m] = 0.0;
            for (long long kk = 0; kk < nk; kk++) {
                long long p = row[C] + kk; int B = pB[p], sB = atom_species[B], nB = bs.norb[sB];
                double R[3]; lattice(cell, pR[3 * p], pR[3 * p + 1], pR[3 * p + 2], R);
                double dB[3] = { r[0] - atom_pos[3 * B] - R[0], r[1] - atom_pos[3 * B + 1] - R[1], r[2] - atom_pos[3 * B + 2] - R[2] };
                if (!phi_eval(&bs, sB, dB, pb)) continue;
                const double *Dp = D + offset[p], *Dm = D + offset[mir[kk]];      /* nC x nB  and  nB x nC */
                for (int mu = 0; mu < nC; mu++) {
                    double t = 0.0;
                    for (int nu = 0; nu < nB; nu++) t += (Dp[mu * nB + nu] + Dm[nu * nC + mu]) * pb[nu];
                    psi[mu] += t;
                }
            }
            double Vg = V[(imod(i, N1) * N2 + imod(j, N2)) * N3 + imod(k, N3)];
            for (int a = 0; a < 3; a++) {
                double s = 0.0;
                for (int mu = 0; mu < nC; mu++) s += gc[3 * mu + a] * psi[mu];
                s *= Vg * dV;
                Fc[a] += s;
                for (int b = 0; b < 3; b++) sg[3 * a + b] -= s * dC[b] / Omega;
            }
        }
        F[3 * C] = Fc[0]; F[3 * C + 1] = Fc[1]; F[3 * C + 2] = Fc[2];
        free(mir);
    }
    if (!sel && sigma) for (int k = 0; k < 9; k++) sigma[k] = sg[k];
    free(row); basis_free(&bs);
    return bad ? -2 : 0;
}
