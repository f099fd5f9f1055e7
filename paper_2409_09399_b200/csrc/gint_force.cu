// gint_force.cu -- Pulay force and stress of the local-potential energy (Eq. 4 and Eq. 5; "for computing forces and
// stresses, the derivatives of the spherical harmonics are also calculated"), fp64, sm_100a.
//
// Reading R15: with E = <D, H> = dV sum_g V_g rho_g, at fixed V (per mesh index), D and dV,
//   F_C^a      = -dE/dtau_C^a = dV sum_g V_g sum_t  grad_a phi_(C,t)(g) . Psi_(C,t)(g),
//   Psi_(C,t)(g) = sum over atom images (B,t') non-zero at g of  ( D_(C,B,t'-t) + D_(B,C,t-t')^T ) phi_(B,t')(g),
//   sigma^{ab} = -(1/Omega) dE/d eps_ab = -(1/Omega) sum_(C,t) dV sum_g V_g ( grad_a phi_(C,t)(g) . Psi_(C,t)(g) ) (r_g - tau_C - t)^b.
// Psi costs what the density costs without the mirror symmetry (every ordered pair of atoms of a batch); the twelve components then
// come from one product each with the orbital gradients -- the order of operations of the paper's force kernels ("same batching,
// orbital gradients, rho_mu_nu contraction").
//
// One CTA per grid batch walks the batch's cubelets (2 x 2 x 2 mesh points) with the neighbour table and activity masks of gint_init:
//   1. phi of the atoms active on the cubelet -> shared memory, [orbital row][8 points];
//   2. Psi rows of those atoms: one thread per orbital row, 8 points in registers, D rows read through L1 from a full-layout copy of
//      D + mirror^T (k_sym_full), phi rows as broadcast 128-bit shared loads;
//   3. gradients of the same atoms at the same points (analytic: spline derivative, gradient of the real harmonics), their products
//      with Psi and V dV: per (atom, point) partial forces in shared memory without atomics, the stress in registers.
// The batch adds 3 doubles per neighbouring atom and 9 for the stress with red.global.add.f64.
#include "gint_internal.h"

#include <mutex>

typedef unsigned long long u64;
namespace {

struct cmaskf { u64 lo, hi; };
__device__ __forceinline__ bool fbit(const cmaskf& m, int i) { return ((i < 64 ? m.lo >> i : m.hi >> (i - 64)) & 1ull) != 0; }

// One warp per public key p: Dfull_p = D_p + D_mirror(p)^T  (both blocks are read; for the on-site key the mirror is the key itself).
__global__ void __launch_bounds__(256) k_sym_full(long long n_pairs, const long long* __restrict__ poff, const int* __restrict__ pcanon,
                                                  const unsigned char* __restrict__ pflag, const int* __restrict__ cpub, const int* __restrict__ cmir,
                                                  const int* __restrict__ pnab, const double* __restrict__ D, double* __restrict__ Dfull) {
    const long long p = (long long)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (p >= n_pairs) return;
    const int lane = threadIdx.x & 31;
    const int c = pcanon[p];
    const int q = pflag[p] ? cmir[c] : cpub[c];
    const int nA = pnab[p] & 0xffff, nB = pnab[p] >> 16;
    const double* d1 = D + poff[p];
    const double* d2 = D + poff[q];             // nB x nA
    double* dst = Dfull + poff[p];
    for (int e = lane; e < nA * nB; e += 32) { const int i = e / nB, j = e - i * nB; dst[e] = d1[e] + d2[j * nA + i]; }
}

struct ForceEntry {
    double x, y, z, rc2;            // image position, cutoff^2
    cmaskf mask;
    int atom, shift, tab_off, n_int, nsh, lpack, row0, norb;
};
struct ForceSmem {
    ForceEntry ent[GINT_MAX_NB];
    int arow[GINT_MAX_NB + 1];      // prefix sums of norb over the atoms active on the current cubelet
    unsigned char act[GINT_MAX_NB];
    int nact;
    double sig[8][9];
};
#define GINT_FORCE_THREADS 256

// radial value and derivative of shell s at r (interval i, b = r/dr - i): cells {y, y'' dr^2/6} of knots i, i + 1
__device__ __forceinline__ void radial2(const double2* __restrict__ row, int nsh, int s, double am, double bb, double inv_dr, double& R, double& R1) {
    const double2 c0 = __ldg(row + s), c1 = __ldg(row + nsh + s);
    R = fma(am, c0.x, fma(bb, c1.x, fma((am * am - 1.0) * am, c0.y, (bb * bb - 1.0) * bb * c1.y)));
    R1 = inv_dr * ((c1.x - c0.x) - (3.0 * am * am - 1.0) * c0.y + (3.0 * bb * bb - 1.0) * c1.y);
}

__global__ void __launch_bounds__(GINT_FORCE_THREADS)
k_force_batch(Geom g, const int* __restrict__ bstart, const NeighEntry* __restrict__ bent,
              const double* __restrict__ atom_pos, const int* __restrict__ atom_spec, const SpeciesDev* __restrict__ sp,
              const double* __restrict__ tab, const int* __restrict__ crow, const u64* __restrict__ ckey, const int* __restrict__ cpub,
              const int* __restrict__ cmir, const long long* __restrict__ poff, const double* __restrict__ V, const double* __restrict__ Dfull,
              double inv_omega, double* __restrict__ F, double* __restrict__ sigma) {
    extern __shared__ __align__(16) unsigned char fsm[];
    ForceSmem& S = *reinterpret_cast<ForceSmem*>(fsm);
    const long long b = blockIdx.x;
    const int e0 = bstart[b], n = bstart[b + 1] - e0;
    if (n == 0) return;
    const int tid = threadIdx.x, lane = tid & 31;
    // dynamic part: pair offsets [n][n], partial forces [n][8][3], phi and Psi [rows][8]
    unsigned* pairp = reinterpret_cast<unsigned*>(fsm + ((sizeof(ForceSmem) + 15) & ~(size_t)15));
    double* facc = reinterpret_cast<double*>(reinterpret_cast<unsigned char*>(pairp) + (((size_t)n * n * 4 + 15) & ~(size_t)15));
    double* phi = facc + (size_t)n * 24;
    const int bz = (int)(b % g.nb[2]), by = (int)((b / g.nb[2]) % g.nb[1]), bx = (int)(b / ((long long)g.nb[2] * g.nb[1]));
    const int i0 = bx * g.bs[0], j0 = by * g.bs[1], k0 = bz * g.bs[2];
    if (tid < n) {
        const NeighEntry e = bent[e0 + tid];
        int t1, t2, t3; unpack_shift(e.shift, t1, t2, t3);
        ForceEntry& E = S.ent[tid];
        image_pos(g, atom_pos + 3 * e.atom, t1, t2, t3, E.x, E.y, E.z);
        const SpeciesDev* Sp = sp + atom_spec[e.atom];
        E.rc2 = Sp->rc * Sp->rc; E.mask = cmaskf{e.mask[0], e.mask[1]};
        E.atom = e.atom; E.shift = e.shift; E.tab_off = Sp->tab_off; E.n_int = Sp->n_int; E.nsh = Sp->n_shell; E.norb = Sp->norb;
        int lp = 0;
        for (int k = 0; k < Sp->n_shell; k++) lp |= Sp->l[k] << (2 * k);
        E.lpack = lp;
    }
    for (int i = tid; i < n * 24; i += GINT_FORCE_THREADS) facc[i] = 0.0;
    __syncthreads();
    if (tid == 0) { int r = 0; for (int e = 0; e < n; e++) { S.ent[e].row0 = r; r += S.ent[e].norb; } }
    // block of (a, b): offset of the public key (atom a, atom b, shift b - shift a) in the full layout, through the canonical key list
    for (int idx = tid; idx < n * n; idx += GINT_FORCE_THREADS) {
        const int a = idx / n, bb = idx - a * n;
        int A = S.ent[a].atom, B = S.ent[bb].atom;
        int ta1, ta2, ta3, tb1, tb2, tb3;
        unpack_shift(S.ent[a].shift, ta1, ta2, ta3); unpack_shift(S.ent[bb].shift, tb1, tb2, tb3);
        int n1 = tb1 - ta1, n2 = tb2 - ta2, n3 = tb3 - ta3;
        const bool ge0 = n1 > 0 || (n1 == 0 && (n2 > 0 || (n2 == 0 && n3 >= 0)));
        bool tr = false;
        if (!(A < B || (A == B && ge0))) { const int t = A; A = B; B = t; n1 = -n1; n2 = -n2; n3 = -n3; tr = true; }
        unsigned off = 0xffffffffu;
        const int m = g.key_m;
        if (abs(n1) <= m && abs(n2) <= m && abs(n3) <= m) {
            const u64 M = (u64)g.key_M;
            const u64 want = (((u64)B * M + (u64)(n1 + m)) * M + (u64)(n2 + m)) * M + (u64)(n3 + m);
            int lo = crow[A], hi = crow[A + 1] - 1;
            while (lo <= hi) {
                const int mid = (lo + hi) >> 1;
                const u64 k = ckey[mid];
                if (k == want) { off = (unsigned)poff[tr ? cmir[mid] : cpub[mid]]; break; }
                if (k < want) lo = mid + 1; else hi = mid - 1;
            }
        }
        pairp[idx] = off;
    }
    __syncthreads();
    const int rows_total = S.ent[n - 1].row0 + S.ent[n - 1].norb;
    double* psi = phi + (size_t)rows_total * 8;
    const double2* tb = reinterpret_cast<const double2*>(tab);
    double sg[9];
#pragma unroll
    for (int k = 0; k < 9; k++) sg[k] = 0.0;
    const int ncx = (min(g.bs[0], g.N[0] - i0) + 1) >> 1, ncy = (min(g.bs[1], g.N[1] - j0) + 1) >> 1, ncz = (min(g.bs[2], g.N[2] - k0) + GINT_CZ - 1) / GINT_CZ;
    for (int cx = 0; cx < ncx; cx++) for (int cy = 0; cy < ncy; cy++) for (int cz = 0; cz < ncz; cz++) {
        const int cl = (cx * 4 + cy) * GINT_NCZ + cz;
        // the atoms active on this cubelet, in list order (warp 0)
        if (tid < 32) {
            int cnt = 0, rows = 0;
            for (int e = lane; e < ((n + 31) & ~31); e += 32) {
                const bool on = e < n && fbit(S.ent[e].mask, cl);
                const unsigned bal = __ballot_sync(0xffffffffu, on);
                const int pos = cnt + __popc(bal & ((1u << lane) - 1u));
                // rows: prefix over the active atoms of their orbital counts
                int no = on ? S.ent[e].norb : 0, inc = no;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
                if (on) { S.act[pos] = (unsigned char)e; S.arow[pos] = rows + inc - no; }
                cnt += __popc(bal);
                rows += __shfl_sync(0xffffffffu, inc, 31);
            }
            if (lane == 0) { S.nact = cnt; S.arow[cnt] = rows; }
        }
        __syncthreads();
        const int nact = S.nact;
        if (nact == 0) { __syncthreads(); continue; }
        // ---- 1. orbital values of the active atoms at the 8 points of the cubelet
        for (int it = tid; it < nact * 8; it += GINT_FORCE_THREADS) {
            const ForceEntry& E = S.ent[S.act[it >> 3]];
            const int p = it & 7;
            const int ix = 2 * cx + (p >> 2), iy = 2 * cy + ((p >> 1) & 1), iz = GINT_CZ * cz + (p & 1);
            double px, py, pz;
            mesh_point(g, i0 + ix, j0 + iy, k0 + iz, px, py, pz);
            const double dx = px - E.x, dy = py - E.y, dz = pz - E.z;
            const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
            const bool inside = r2 < E.rc2;
            const double r = sqrt(fmin(r2, E.rc2));
            const bool tiny = r < 1e-12;
            const double ir = tiny ? 0.0 : 1.0 / r;
            const double x = r * g.inv_dr;
            const int i = min((int)x, E.n_int - 1);
            const double bb = x - (double)i, am = 1.0 - bb;
            const double2* row = tb + (E.tab_off + i * E.nsh);
            const double ux = dx * ir, uy = dy * ir, uz = dz * ir;
            const double w0 = inside ? 1.0 : 0.0;
            double* o = phi + (size_t)E.row0 * 8 + p;
            for (int s = 0; s < E.nsh; s++) {
                double R, R1; radial2(row, E.nsh, s, am, bb, g.inv_dr, R, R1);
                R *= w0;
                const int l = (E.lpack >> (2 * s)) & 3;
                if (l == 0) { o[0] = 0.28209479177387814 * R; o += 8; }
                else if (l == 1) {
                    const double c = 0.4886025119029199 * R;
                    o[0] = c * uy; o[8] = c * uz; o[16] = c * ux; o += 24;
                } else {
                    const double c = 1.0925484305920792 * R;
                    o[0] = c * ux * uy; o[8] = c * uy * uz; o[16] = (tiny ? 0.0 : 0.31539156525252005) * R * fma(3.0 * uz, uz, -1.0);
                    o[24] = c * ux * uz; o[32] = 0.5462742152960396 * R * fma(ux, ux, -uy * uy); o += 40;
                }
            }
        }
        __syncthreads();
        // ---- 2. Psi rows of the active atoms: Psi_a[i][p] = sum_b sum_j Dfull_(a,b)[i][j] phi_b[j][p]
        const int nrows = S.arow[nact];
        for (int rr = tid; rr < nrows; rr += GINT_FORCE_THREADS) {
            int lo = 0, hi = nact - 1;
            while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (S.arow[mid] <= rr) lo = mid; else hi = mid - 1; }
            const int a = S.act[lo], i = rr - S.arow[lo], nA = S.ent[a].norb;
            double acc[8];
#pragma unroll
            for (int p = 0; p < 8; p++) acc[p] = 0.0;
            for (int kb = 0; kb < nact; kb++) {
                const int bb = S.act[kb];
                // Dfull_(a,b)[i][j] is read as Dfull_(b,a)[j][i] (the full-layout copy is symmetric: Dfull_q = Dfull_p^T for mirror keys):
                // the threads of a warp hold consecutive rows i, so that their loads fall into a few sectors instead of one each
                const unsigned off = pairp[bb * n + a];
                if (off == 0xffffffffu) continue;
                const int nB = S.ent[bb].norb;
                const double* dcol = Dfull + off + i;
                const double2* pr = reinterpret_cast<const double2*>(phi + (size_t)S.ent[bb].row0 * 8);
                for (int j = 0; j < nB; j++) {
                    const double d = __ldg(dcol + (size_t)j * nA);
                    const double2 f0 = pr[4 * j], f1 = pr[4 * j + 1], f2 = pr[4 * j + 2], f3 = pr[4 * j + 3];
                    acc[0] = fma(d, f0.x, acc[0]); acc[1] = fma(d, f0.y, acc[1]); acc[2] = fma(d, f1.x, acc[2]); acc[3] = fma(d, f1.y, acc[3]);
                    acc[4] = fma(d, f2.x, acc[4]); acc[5] = fma(d, f2.y, acc[5]); acc[6] = fma(d, f3.x, acc[6]); acc[7] = fma(d, f3.y, acc[7]);
                }
            }
            double2* out = reinterpret_cast<double2*>(psi + (size_t)(S.ent[a].row0 + i) * 8);
            out[0] = make_double2(acc[0], acc[1]); out[1] = make_double2(acc[2], acc[3]); out[2] = make_double2(acc[4], acc[5]); out[3] = make_double2(acc[6], acc[7]);
        }
        __syncthreads();
        // ---- 3. gradients of the active atoms at the same points, times Psi and V dV
        for (int it = tid; it < nact * 8; it += GINT_FORCE_THREADS) {
            const int e = S.act[it >> 3];
            const ForceEntry& E = S.ent[e];
            const int p = it & 7;
            const int ix = 2 * cx + (p >> 2), iy = 2 * cy + ((p >> 1) & 1), iz = GINT_CZ * cz + (p & 1);
            const int gi = i0 + ix, gj = j0 + iy, gk = k0 + iz;
            const bool in_batch = ix < g.bs[0] && iy < g.bs[1] && iz < g.bs[2] && gi < g.N[0] && gj < g.N[1] && gk < g.N[2];
            double px, py, pz;
            mesh_point(g, gi, gj, gk, px, py, pz);
            const double dx = px - E.x, dy = py - E.y, dz = pz - E.z;
            const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
            if (!(in_batch && r2 < E.rc2)) continue;
            const double w = __ldg(V + ((size_t)gi * g.N[1] + gj) * g.N[2] + gk) * g.dV;
            const double r = sqrt(r2);
            const bool tiny = r < 1e-12;
            const double ir = tiny ? 0.0 : 1.0 / r;
            const double x = r * g.inv_dr;
            const int i = min((int)x, E.n_int - 1);
            const double bb = x - (double)i, am = 1.0 - bb;
            const double2* row = tb + (E.tab_off + i * E.nsh);
            const double u[3] = {dx * ir, dy * ir, dz * ir};
            const double* ps = psi + (size_t)E.row0 * 8 + p;
            double s3[3] = {0.0, 0.0, 0.0};
            for (int s = 0; s < E.nsh; s++) {
                double R, R1; radial2(row, E.nsh, s, am, bb, g.inv_dr, R, R1);
                const int l = (E.lpack >> (2 * s)) & 3;
                // grad phi = (R' - l R / r) u c P(u) + (R / r) c grad_u P(u); at the nucleus: 0, except c_1 R'(0) e_m for l = 1
                if (l == 0) {
                    const double t = 0.28209479177387814 * R1 * ps[0];
#pragma unroll
                    for (int a = 0; a < 3; a++) s3[a] = fma(t, u[a], s3[a]);
                    ps += 8;
                } else if (l == 1) {
                    const double c = 0.4886025119029199;
                    const double A = tiny ? 0.0 : c * (R1 - R * ir), Bq = tiny ? c * R1 : c * R * ir;
                    const double P[3] = {u[1], u[2], u[0]};
                    const int ax[3] = {1, 2, 0};
#pragma unroll
                    for (int m = 0; m < 3; m++) {
                        const double q = ps[8 * m];
#pragma unroll
                        for (int a = 0; a < 3; a++) s3[a] = fma(q, A * P[m] * u[a] + (a == ax[m] ? Bq : 0.0), s3[a]);
                    }
                    ps += 24;
                } else {
                    const double c2 = 1.0925484305920792;
                    const double cm[5] = {c2, c2, 0.31539156525252005, c2, 0.5462742152960396};
                    const double P[5] = {u[0] * u[1], u[1] * u[2], 2.0 * u[2] * u[2] - u[0] * u[0] - u[1] * u[1], u[0] * u[2], u[0] * u[0] - u[1] * u[1]};
                    const double G[5][3] = {{u[1], u[0], 0.0}, {0.0, u[2], u[1]}, {-2.0 * u[0], -2.0 * u[1], 4.0 * u[2]}, {u[2], 0.0, u[0]}, {2.0 * u[0], -2.0 * u[1], 0.0}};
                    const double A = tiny ? 0.0 : (R1 - 2.0 * R * ir), Bq = tiny ? 0.0 : R * ir;
#pragma unroll
                    for (int m = 0; m < 5; m++) {
                        const double q = ps[8 * m] * cm[m];
#pragma unroll
                        for (int a = 0; a < 3; a++) s3[a] = fma(q, A * P[m] * u[a] + Bq * G[m][a], s3[a]);
                    }
                    ps += 40;
                }
            }
            const double d3[3] = {dx, dy, dz};
            double* fa = facc + ((size_t)e * 8 + p) * 3;
#pragma unroll
            for (int a = 0; a < 3; a++) {
                const double sa = w * s3[a];
                fa[a] += sa;
#pragma unroll
                for (int bq = 0; bq < 3; bq++) sg[3 * a + bq] = fma(sa, d3[bq], sg[3 * a + bq]);
            }
        }
        __syncthreads();
    }
    // ---- the batch's contribution: 3 adds per neighbouring atom, 9 for the stress
    for (int idx = tid; idx < n * 3; idx += GINT_FORCE_THREADS) {
        const int e = idx / 3, a = idx - 3 * e;
        double v = 0.0;
#pragma unroll
        for (int p = 0; p < 8; p++) v += facc[((size_t)e * 8 + p) * 3 + a];
        if (v != 0.0) atomicAdd(F + 3 * (size_t)S.ent[e].atom + a, v);
    }
#pragma unroll
    for (int k = 0; k < 9; k++) {
        double v = sg[k];
        for (int d = 16; d; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
        if (lane == 0) S.sig[tid >> 5][k] = v;
    }
    __syncthreads();
    if (tid < 9 && sigma) {
        double v = 0.0;
        for (int w = 0; w < GINT_FORCE_THREADS / 32; w++) v += S.sig[w][tid];
        if (v != 0.0) atomicAdd(sigma + tid, -v * inv_omega);
    }
}

}  // namespace

size_t gint_force_smem(const gint_ctx* c) {
    const size_t n = (size_t)c->geom.max_nb, rows = (size_t)c->geom.max_cols;
    return ((sizeof(ForceSmem) + 15) & ~(size_t)15) + ((n * n * 4 + 15) & ~(size_t)15) + n * 24 * sizeof(double) + 2 * rows * 8 * sizeof(double);
}

int gint_launch_force(gint_ctx* c, const double* V, const double* D, double* F, double* sigma, cudaStream_t st) {
    GINT_CUDA(cudaSetDevice(c->device));
    GINT_CUDA(cudaMemsetAsync(F, 0, sizeof(double) * 3 * (size_t)c->n_atoms, st));
    if (sigma) GINT_CUDA(cudaMemsetAsync(sigma, 0, sizeof(double) * 9, st));
    if (c->n_batch == 0 || c->n_values == 0) return GINT_OK;
    if (c->n_values >= (1ll << 32)) GINT_FAIL(GINT_ERR_UNSUPPORTED, "gint_force_stress: more than 2^32 matrix elements");
    const size_t smem = gint_force_smem(c);
    if (smem > c->smem_optin)
        GINT_FAIL(GINT_ERR_UNSUPPORTED, "gint_force_stress: a batch of %d atom images and %d orbitals needs %zu bytes of shared memory (limit %zu); "
                  "initialise with GINT_FLAG_FORCE, or a smaller GINT_FLAG_BATCH", c->geom.max_nb, c->geom.max_cols, smem, c->smem_optin);
    if (!c->d_dfull) {
        GINT_CUDA(cudaMalloc((void**)&c->d_dfull, sizeof(double) * (size_t)c->n_values));
        c->device_bytes += sizeof(double) * (size_t)c->n_values;
    }
    if (!c->force_configured) {      // once per context, not per call
        GINT_CUDA(cudaFuncSetAttribute(k_force_batch, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem_optin));
        c->force_configured = true;
    }
    GINT_CUDA(cudaEventRecord(c->ev_force[0], st));
    k_sym_full<<<(unsigned)((c->n_pairs + 7) / 8), 256, 0, st>>>(c->n_pairs, c->d_poff, c->d_pcanon, c->d_pflag, c->d_cpub, c->d_cmir, c->d_pnA, D, c->d_dfull);
    GINT_CUDA(cudaGetLastError());
    const double omega = c->geom.dV * (double)c->geom.N[0] * c->geom.N[1] * c->geom.N[2];
    k_force_batch<<<(unsigned)c->n_batch_total, GINT_FORCE_THREADS, smem, st>>>(c->geom, c->d_bstart, c->d_bent, c->d_atom_pos, c->d_atom_species,
        c->d_species, c->d_tab, c->d_crow, c->d_ckey, c->d_cpub, c->d_cmir, c->d_poff, V, c->d_dfull, 1.0 / omega, F, sigma);
    GINT_CUDA(cudaGetLastError());
    GINT_CUDA(cudaEventRecord(c->ev_force[1], st));
    c->timed_force = true;
    return GINT_OK;
}

// ================================================================================================================================
// gint_force_stress_static -- the same two kernels as gint_force_stress, for callers that must not allocate device memory.
//
// gint_force_stress needs one piece of scratch: Dfull = D + mirror^T in the pair-list layout (8 * n_values bytes), which it obtains
// with cudaMalloc on its first call.  Some callers cannot afford that call: a DFT driver that handed the whole device to its own
// arena at start-up (a cudaMalloc then fails although "its" memory is free), a job inside a fixed-size MPS / MIG memory slice, or an
// ionic-step loop that must not hit cudaMalloc's device-wide synchronisation while other streams are busy.  For them the scratch
// lives in the library image itself: the array below is part of libgint.so's device data, so every GPU on which the library's
// module gets loaded holds these GINT_STATIC_SCRATCH_DOUBLES * 8 bytes = 8 MiB until the process exits, whether or not this entry
// point is ever called.  That is why the limit is small; systems beyond it use gint_force_stress.
//
// The array is shared by every context and every call on a device, and nothing serialises them: two calls that can run at the same
// time on the GPU (two streams, two contexts, two host threads) overwrite each other's Dfull.  Order such calls on one stream.
// Nothing in it has to start at zero: k_sym_full writes every element of [0, n_values) before k_force_batch reads any of them, so
// the previous call's contents (another geometry's, perhaps) are never seen.  F and sigma, the outputs, are cleared as usual.
static __device__ __align__(256) double g_dfull_static[GINT_STATIC_SCRATCH_DOUBLES];

namespace {
// Per-device set-up, done by the first call on that device: in host code `g_dfull_static` names a host-side shadow of the symbol,
// not device memory, so the address the kernels get has to come from cudaGetSymbolAddress (asked with that device current).
struct StaticSetup { bool done = false; double* dfull = nullptr; int smem_optin = 0; };
constexpr int kMaxDevices = 64;
StaticSetup g_static_setup[kMaxDevices];
std::mutex g_static_mutex;

int static_setup(int device, const StaticSetup** out) {
    if (device < 0 || device >= kMaxDevices) GINT_FAIL(GINT_ERR_UNSUPPORTED, "gint_force_stress_static: device ordinal %d (supported: 0..%d)", device, kMaxDevices - 1);
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticSetup& s = g_static_setup[device];
    if (!s.done) {
        GINT_CUDA(cudaSetDevice(device));
        void* p = nullptr;
        GINT_CUDA(cudaGetSymbolAddress(&p, g_dfull_static));
        if (!p || ((uintptr_t)p & 255)) GINT_FAIL(GINT_ERR_CUDA, "gint_force_stress_static: bad address %p for the static scratch", p);
        GINT_CUDA(cudaDeviceGetAttribute(&s.smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device));
        GINT_CUDA(cudaFuncSetAttribute(k_force_batch, cudaFuncAttributeMaxDynamicSharedMemorySize, s.smem_optin));
        s.dfull = static_cast<double*>(p);
        s.done = true;
    }
    *out = &s;
    return GINT_OK;
}
}  // namespace

extern "C" int gint_force_stress_static(gint_ctx* c, const double* V_dev, const double* D_dev, double* F_dev, double* sigma_dev, void* stream) {
    if (!c) GINT_FAIL(GINT_ERR_BAD_STATE, "NULL context");
    if (!V_dev || (!D_dev && c->n_values) || (!F_dev && c->n_atoms)) GINT_FAIL(GINT_ERR_INVALID_ARG, "NULL device pointer");
    if (((uintptr_t)V_dev | (uintptr_t)D_dev | (uintptr_t)F_dev | (uintptr_t)sigma_dev) & 7) GINT_FAIL(GINT_ERR_INVALID_ARG, "device pointers must be 8-byte aligned");
    if (c->n_values > (long long)GINT_STATIC_SCRATCH_DOUBLES)
        GINT_FAIL(GINT_ERR_UNSUPPORTED, "gint_force_stress_static: the pair list holds %lld matrix elements, the static scratch %lld "
                  "(GINT_STATIC_SCRATCH_DOUBLES); use gint_force_stress, which allocates its own", c->n_values, (long long)GINT_STATIC_SCRATCH_DOUBLES);
    DeviceGuard guard;
    const StaticSetup* s = nullptr;
    if (int rc = static_setup(c->device, &s)) return rc;
    GINT_CUDA(cudaSetDevice(c->device));
    cudaStream_t st = (cudaStream_t)stream;
    GINT_CUDA(cudaMemsetAsync(F_dev, 0, sizeof(double) * 3 * (size_t)c->n_atoms, st));
    if (sigma_dev) GINT_CUDA(cudaMemsetAsync(sigma_dev, 0, sizeof(double) * 9, st));
    if (c->n_batch == 0 || c->n_values == 0) return GINT_OK;
    const size_t smem = gint_force_smem(c);
    if (smem > (size_t)s->smem_optin) GINT_FAIL(GINT_ERR_UNSUPPORTED, "gint_force_stress_static: a batch of %d orbitals needs %zu bytes of shared memory", c->geom.max_cols, smem);
    GINT_CUDA(cudaEventRecord(c->ev_force[0], st));
    k_sym_full<<<(unsigned)((c->n_pairs + 7) / 8), 256, 0, st>>>(c->n_pairs, c->d_poff, c->d_pcanon, c->d_pflag, c->d_cpub, c->d_cmir, c->d_pnA, D_dev, s->dfull);
    GINT_CUDA(cudaGetLastError());
    const double omega = c->geom.dV * (double)c->geom.N[0] * c->geom.N[1] * c->geom.N[2];
    k_force_batch<<<(unsigned)c->n_batch_total, GINT_FORCE_THREADS, smem, st>>>(c->geom, c->d_bstart, c->d_bent, c->d_atom_pos, c->d_atom_species,
        c->d_species, c->d_tab, c->d_crow, c->d_ckey, c->d_cpub, c->d_cmir, c->d_poff, V_dev, s->dfull, 1.0 / omega, F_dev, sigma_dev);
    GINT_CUDA(cudaGetLastError());
    GINT_CUDA(cudaEventRecord(c->ev_force[1], st));
    c->timed_force = true;
    return GINT_OK;
}
