// gint_kernels.cu -- the per-call hot path (north_star steps 2 and 3), fp64, sm_100a.
//
// One CTA processes one grid batch: it evaluates the orbitals of the batch's neighbouring atom
// images into shared memory (the paper's orbital-value kernel, but never written to global
// memory), then contracts them on the FP64 tensor pipe (mma.sync m8n8k4 f64 = DMMA):
//   vlocal:  W = Phi^T diag(V dV) Phi           (Eq. 2)  -> canonical-half H blocks
//   rho:     rho_g = sum_{ij} Phi_gi D_ij Phi_gj (Eq. 3)  -> one plain store per mesh point
// Only one of each mirror pair of blocks, (A,B,n) / (B,A,-n), is computed ("canonical half"); small
// streaming kernels convert between the public pair-list layout and the canonical layout.
#include "gint_internal.h"

// ---------------------------------------------------------------------------------------------------
// shared-memory carve-up (bytes), identical on host and device
struct SmemLayout {
    unsigned phi, pts, vw, epos, eatom, espec, eshift, colstart, colslot, boff, total;
};
__host__ __device__ inline SmemLayout smem_layout(const Geom& g) {
    SmemLayout L;
    const unsigned cols_pad = (unsigned)((g.max_cols + 7) / 8 * 8);
    const unsigned Kp = (unsigned)(g.LD - 4);
    unsigned o = 0;
    L.phi = o; o += cols_pad * (unsigned)g.LD * 8u;
    L.pts = o; o += 3u * Kp * 8u;
    L.vw = o; o += Kp * 8u;
    L.epos = o; o += 3u * (unsigned)g.max_nb * 8u;
    L.eatom = o; o += (unsigned)g.max_nb * 4u;
    L.espec = o; o += (unsigned)g.max_nb * 4u;
    L.eshift = o; o += (unsigned)g.max_nb * 4u;
    L.colstart = o; o += ((unsigned)g.max_nb + 1u) * 4u;
    L.boff = o; o += (unsigned)g.max_nb * (unsigned)g.max_nb * 4u;
    L.colslot = o; o += (cols_pad + 7u) / 8u * 8u;
    L.total = (o + 15u) / 16u * 16u;
    return L;
}
size_t gint_smem_needed(const Geom& g) { return smem_layout(g).total; }

// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

struct BatchView {
    int i0, j0, k0, ex, ey, ez, Kb, Kp;   // origin, extents, points, points padded to a multiple of 8
    int nbr, ncols, nfrag;                // neighbour entries, orbitals, 8-wide column fragments
};

// Everything a batch needs before the orbital evaluation: neighbour entries, image positions, column map,
// canonical block offsets of every slot pair a <= b, mesh-point coordinates.
__device__ __forceinline__ void load_batch(const Geom& g, const SmemLayout& L, unsigned char* smem, int b, BatchView& bv,
                                           const int* __restrict__ bstart, const NeighEntry* __restrict__ bent,
                                           const double* __restrict__ atom_pos, const int* __restrict__ atom_spec,
                                           const SpeciesDev* __restrict__ sp, const int* __restrict__ crow,
                                           const unsigned long long* __restrict__ ckey, const unsigned int* __restrict__ coff) {
    double* s_pts = (double*)(smem + L.pts);
    double* s_epos = (double*)(smem + L.epos);
    int* s_atom = (int*)(smem + L.eatom);
    int* s_spec = (int*)(smem + L.espec);
    int* s_shift = (int*)(smem + L.eshift);
    int* s_colstart = (int*)(smem + L.colstart);
    unsigned char* s_colslot = smem + L.colslot;
    unsigned int* s_boff = (unsigned int*)(smem + L.boff);
    const int tid = threadIdx.x, nt = blockDim.x;

    const int bz = b % g.nb[2], by = (b / g.nb[2]) % g.nb[1], bx = b / (g.nb[2] * g.nb[1]);
    bv.i0 = bx * g.bs[0]; bv.j0 = by * g.bs[1]; bv.k0 = bz * g.bs[2];
    bv.ex = min(g.bs[0], g.N[0] - bv.i0); bv.ey = min(g.bs[1], g.N[1] - bv.j0); bv.ez = min(g.bs[2], g.N[2] - bv.k0);
    bv.Kb = bv.ex * bv.ey * bv.ez; bv.Kp = (bv.Kb + 7) & ~7;
    const int e0 = bstart[b];
    bv.nbr = bstart[b + 1] - e0;

    if (tid < bv.nbr) {
        NeighEntry e = bent[e0 + tid];
        int t1, t2, t3; unpack_shift(e.shift, t1, t2, t3);
        s_atom[tid] = e.atom; s_shift[tid] = e.shift; s_spec[tid] = atom_spec[e.atom];
        s_epos[3 * tid + 0] = atom_pos[3 * e.atom + 0] + t1 * g.a[0] + t2 * g.a[3] + t3 * g.a[6];
        s_epos[3 * tid + 1] = atom_pos[3 * e.atom + 1] + t1 * g.a[1] + t2 * g.a[4] + t3 * g.a[7];
        s_epos[3 * tid + 2] = atom_pos[3 * e.atom + 2] + t1 * g.a[2] + t2 * g.a[5] + t3 * g.a[8];
    }
    if (tid >= 64 && tid < 64 + bv.Kp) {           // mesh points (a different warp range than the entry loads)
        const int q = tid - 64;
        double x = 0, y = 0, z = 0;
        if (q < bv.Kb) {
            int qk = q % bv.ez, qj = (q / bv.ez) % bv.ey, qi = q / (bv.ez * bv.ey);
            mesh_point(g, bv.i0 + qi, bv.j0 + qj, bv.k0 + qk, x, y, z);
        }
        s_pts[3 * q] = x; s_pts[3 * q + 1] = y; s_pts[3 * q + 2] = z;
    }
    __syncthreads();
    if (tid < 32) {                                  // column starts: warp scan over the entries' orbital counts
        int carry = 0;
        for (int s0 = 0; s0 < bv.nbr; s0 += 32) {
            int s = s0 + tid;
            int v = s < bv.nbr ? sp[s_spec[s]].norb : 0, inc = v;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { int t = __shfl_up_sync(0xffffffffu, inc, d); if (tid >= d) inc += t; }
            if (s < bv.nbr) s_colstart[s] = carry + inc - v;
            carry += __shfl_sync(0xffffffffu, inc, 31);
        }
        if (tid == 0) s_colstart[bv.nbr] = carry;
    }
    __syncthreads();
    bv.ncols = s_colstart[bv.nbr];
    bv.nfrag = (bv.ncols + 7) >> 3;
    for (int c = tid; c < bv.nfrag * 8; c += nt) {   // column -> slot (binary search in colstart)
        int slot = 255;
        if (c < bv.ncols) {
            int lo = 0, hi = bv.nbr - 1;
            while (lo < hi) { int mid = (lo + hi + 1) >> 1; if (s_colstart[mid] <= c) lo = mid; else hi = mid - 1; }
            slot = lo;
        }
        s_colslot[c] = (unsigned char)slot;
    }
    for (int idx = tid; idx < bv.nbr * bv.nbr; idx += nt) {   // canonical block of slot pair (a <= b)
        const int a = idx / bv.nbr, bb = idx - a * bv.nbr;
        unsigned int off = 0xffffffffu;
        if (a <= bb) {
            int ta1, ta2, ta3, tb1, tb2, tb3;
            unpack_shift(s_shift[a], ta1, ta2, ta3); unpack_shift(s_shift[bb], tb1, tb2, tb3);
            const int n1 = tb1 - ta1, n2 = tb2 - ta2, n3 = tb3 - ta3, m = g.key_m;
            if (abs(n1) <= m && abs(n2) <= m && abs(n3) <= m) {
                const unsigned long long M = (unsigned long long)g.key_M;
                const unsigned long long want = (((unsigned long long)s_atom[bb] * M + (unsigned long long)(n1 + m)) * M + (unsigned long long)(n2 + m)) * M + (unsigned long long)(n3 + m);
                int lo = crow[s_atom[a]], hi = crow[s_atom[a] + 1] - 1;
                while (lo <= hi) {
                    int mid = (lo + hi) >> 1;
                    unsigned long long k = ckey[mid];
                    if (k == want) { off = coff[mid]; break; }
                    if (k < want) lo = mid + 1; else hi = mid - 1;
                }
            }
        }
        s_boff[a * g.max_nb + bb] = off;
    }
}

// Orbital values of the batch (north_star step 2): Phi[col][q] = R_s(|d|) Y_lm(d/|d|), zero for |d| >= rc
// (Fig. 6).  One work item = (mesh point q, neighbour slot s); q runs fastest so a
// warp writes consecutive shared-memory words.  Radial part: per-interval cubic in b = r/dr - i (reading R5).
__device__ __forceinline__ void eval_phi(const Geom& g, const SmemLayout& L, unsigned char* smem, const BatchView& bv,
                                         const SpeciesDev* __restrict__ sp, const double* __restrict__ tab) {
    double* s_phi = (double*)(smem + L.phi);
    const double* s_pts = (const double*)(smem + L.pts);
    const double* s_epos = (const double*)(smem + L.epos);
    const int* s_spec = (const int*)(smem + L.espec);
    const int* s_colstart = (const int*)(smem + L.colstart);
    const int LD = g.LD;
    const int items = bv.Kp * bv.nbr;
    for (int idx = threadIdx.x; idx < items; idx += blockDim.x) {
        const int s = idx / bv.Kp, q = idx - s * bv.Kp;
        const SpeciesDev* S = sp + s_spec[s];
        double* out = s_phi + s_colstart[s] * LD + q;
        const int norb = S->norb;
        bool inside = false;
        double dx = 0, dy = 0, dz = 0, r = 0;
        if (q < bv.Kb) {
            dx = s_pts[3 * q] - s_epos[3 * s]; dy = s_pts[3 * q + 1] - s_epos[3 * s + 1]; dz = s_pts[3 * q + 2] - s_epos[3 * s + 2];
            r = sqrt(dx * dx + dy * dy + dz * dz);
            inside = r < S->rc;
        }
        if (!inside) {
            for (int o = 0; o < norb; o++) out[o * LD] = 0.0;
            continue;
        }
        const double x = r * g.inv_dr;
        int i = (int)x;
        i = min(i, S->n_int - 1);
        const double bq = x - (double)i;
        const int nsh = S->n_shell;
        const double2* row = reinterpret_cast<const double2*>(tab) + ((size_t)S->tab_off + (size_t)i * nsh) * 2;
        const bool tiny = r < 1e-12;
        const double ir = tiny ? 0.0 : 1.0 / r;
        const double ux = dx * ir, uy = dy * ir, uz = dz * ir;
        int o = 0;
        for (int k = 0; k < nsh; k++) {
            const double2 c01 = __ldg(row + 2 * k), c23 = __ldg(row + 2 * k + 1);
            double R = fma(fma(fma(c23.y, bq, c23.x), bq, c01.y), bq, c01.x);
            const int l = S->l[k];
            if (l == 0) {
                out[(o++) * LD] = R * 0.28209479177387814;
            } else if (l == 1) {
                R = tiny ? 0.0 : R * 0.4886025119029199;
                out[(o++) * LD] = R * uy; out[(o++) * LD] = R * uz; out[(o++) * LD] = R * ux;
            } else {
                R = tiny ? 0.0 : R;
                const double c2 = R * 1.0925484305920792;
                out[(o++) * LD] = c2 * ux * uy;
                out[(o++) * LD] = c2 * uy * uz;
                out[(o++) * LD] = R * 0.31539156525252005 * (3.0 * uz * uz - 1.0);
                out[(o++) * LD] = c2 * ux * uz;
                out[(o++) * LD] = R * 0.5462742152960396 * (ux * ux - uy * uy);
            }
        }
    }
    // zero the padding columns ncols .. 8*nfrag-1
    const int padc = bv.nfrag * 8 - bv.ncols;
    for (int idx = threadIdx.x; idx < padc * bv.Kp; idx += blockDim.x) {
        const int c = bv.ncols + idx / bv.Kp, q = idx % bv.Kp;
        s_phi[c * LD + q] = 0.0;
    }
}

// tile t of the upper block triangle: row block I (4 fragments = 32 orbitals), column pair J (2 fragments = 16
// orbitals), J >= 2I.  Returns false when t is past the last tile.
__device__ __forceinline__ bool decode_tile(int t, int nfrag, int& I, int& J) {
    const int nrb = (nfrag + 3) >> 2, ncb = (nfrag + 1) >> 1;
    for (I = 0; I < nrb; I++) {
        const int w = ncb - 2 * I;
        if (t < w) { J = 2 * I + t; return true; }
        t -= w;
    }
    return false;
}

// ---------------------------------------------------------------------------------------------------
// gint_vlocal main kernel (north_star step 3a): W = Phi^T diag(V dV) Phi per batch, upper block triangle only,
// accumulated into the canonical-half value array with fp64 reductions (red.global.add.f64).
__global__ void __launch_bounds__(GINT_THREADS, 1)
k_vlocal(Geom g, const int* __restrict__ order, const int* __restrict__ bstart, const NeighEntry* __restrict__ bent,
         const double* __restrict__ atom_pos, const int* __restrict__ atom_spec, const SpeciesDev* __restrict__ sp,
         const double* __restrict__ tab, const int* __restrict__ crow, const unsigned long long* __restrict__ ckey,
         const unsigned int* __restrict__ coff, const double* __restrict__ V, double* __restrict__ Hc) {
    extern __shared__ __align__(16) unsigned char smem[];
    const SmemLayout L = smem_layout(g);
    BatchView bv;
    const int b = order[blockIdx.x];
    load_batch(g, L, smem, b, bv, bstart, bent, atom_pos, atom_spec, sp, crow, ckey, coff);
    double* s_vw = (double*)(smem + L.vw);
    if ((int)threadIdx.x < bv.Kp) {
        const int q = threadIdx.x;
        double v = 0.0;
        if (q < bv.Kb) {
            int qk = q % bv.ez, qj = (q / bv.ez) % bv.ey, qi = q / (bv.ez * bv.ey);
            v = V[((size_t)(bv.i0 + qi) * g.N[1] + (bv.j0 + qj)) * g.N[2] + (bv.k0 + qk)] * g.dV;
        }
        s_vw[q] = v;
    }
    __syncthreads();
    eval_phi(g, L, smem, bv, sp, tab);
    __syncthreads();

    const double* s_phi = (const double*)(smem + L.phi);
    const int* s_colstart = (const int*)(smem + L.colstart);
    const unsigned char* s_colslot = smem + L.colslot;
    const unsigned int* s_boff = (const unsigned int*)(smem + L.boff);
    const int LD = g.LD, lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const int lr = lane >> 2, lc = lane & 3;
    const int ksteps = bv.Kp >> 2;

    for (int t = warp;; t += nwarp) {
        int I, J;
        if (!decode_tile(t, bv.nfrag, I, J)) break;
        const int fr0 = 4 * I, fc0 = 2 * J;
        const int nmi = min(4, bv.nfrag - fr0), nnj = min(2, bv.nfrag - fc0);
        double acc[4][2][2];
#pragma unroll
        for (int mi = 0; mi < 4; mi++)
#pragma unroll
            for (int nj = 0; nj < 2; nj++) { acc[mi][nj][0] = 0.0; acc[mi][nj][1] = 0.0; }
        const double* pa = s_phi + ((fr0 * 8 + lr) * LD + lc);
        const double* pb = s_phi + ((fc0 * 8 + lr) * LD + lc);
        for (int ks = 0; ks < ksteps; ks++) {
            const double w = s_vw[4 * ks + lc];
            double a[4], bf[2];
#pragma unroll
            for (int mi = 0; mi < 4; mi++) a[mi] = mi < nmi ? pa[mi * 8 * LD + 4 * ks] : 0.0;
#pragma unroll
            for (int nj = 0; nj < 2; nj++) bf[nj] = nj < nnj ? pb[nj * 8 * LD + 4 * ks] * w : 0.0;
#pragma unroll
            for (int mi = 0; mi < 4; mi++)
#pragma unroll
                for (int nj = 0; nj < 2; nj++) dmma884(acc[mi][nj][0], acc[mi][nj][1], a[mi], bf[nj]);
        }
        // flush: element (i, j) belongs to slot pair (sa, sb); keep sa < sb, and i <= j inside a diagonal block
#pragma unroll
        for (int nj = 0; nj < 2; nj++) {
#pragma unroll
            for (int e = 0; e < 2; e++) {
                const int j = (fc0 + nj) * 8 + 2 * lc + e;
                if (nj >= nnj) continue;
                const int sb = s_colslot[j];
                if (sb == 255) continue;
                const int cb = s_colstart[sb], nB = s_colstart[sb + 1] - cb, ob = j - cb;
#pragma unroll
                for (int mi = 0; mi < 4; mi++) {
                    if (mi >= nmi) continue;
                    const int i = (fr0 + mi) * 8 + lr;
                    const int sa = s_colslot[i];
                    if (sa > sb || (sa == sb && i > j)) continue;     // sa == 255 is caught by sa > sb
                    const unsigned int off = s_boff[sa * g.max_nb + sb];
                    if (off == 0xffffffffu) continue;
                    const int oa = i - s_colstart[sa];
                    const double val = acc[mi][nj][e];
                    atomicAdd(Hc + off + oa * nB + ob, val);
                    if (sa == sb && i < j) atomicAdd(Hc + off + ob * nB + oa, val);
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// gint_rho main kernel (north_star step 3b): rho_g = sum over the same upper-triangle tiles of
// rowsum( (Phi[:, I] Dh[I, J]) o Phi[:, J] ), Dh = canonical-half, symmetrised density blocks (k_sym_D).
__global__ void __launch_bounds__(GINT_THREADS, 1)
k_rho(Geom g, const int* __restrict__ order, const int* __restrict__ bstart, const NeighEntry* __restrict__ bent,
      const double* __restrict__ atom_pos, const int* __restrict__ atom_spec, const SpeciesDev* __restrict__ sp,
      const double* __restrict__ tab, const int* __restrict__ crow, const unsigned long long* __restrict__ ckey,
      const unsigned int* __restrict__ coff, const double* __restrict__ Dh, double* __restrict__ rho) {
    extern __shared__ __align__(16) unsigned char smem[];
    const SmemLayout L = smem_layout(g);
    BatchView bv;
    const int b = order[blockIdx.x];
    load_batch(g, L, smem, b, bv, bstart, bent, atom_pos, atom_spec, sp, crow, ckey, coff);
    double* s_rho = (double*)(smem + L.vw);
    if ((int)threadIdx.x < bv.Kp) s_rho[threadIdx.x] = 0.0;
    __syncthreads();
    eval_phi(g, L, smem, bv, sp, tab);
    __syncthreads();

    const double* s_phi = (const double*)(smem + L.phi);
    const int* s_colstart = (const int*)(smem + L.colstart);
    const unsigned char* s_colslot = smem + L.colslot;
    const unsigned int* s_boff = (const unsigned int*)(smem + L.boff);
    const int LD = g.LD, lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const int lr = lane >> 2, lc = lane & 3;
    const int mfrag = bv.Kp >> 3;

    for (int m0 = 0; m0 < mfrag; m0 += 8) {
        const int nmf = min(8, mfrag - m0);
        double part[8];
#pragma unroll
        for (int mf = 0; mf < 8; mf++) part[mf] = 0.0;
        for (int t = warp;; t += nwarp) {
            int I, J;
            if (!decode_tile(t, bv.nfrag, I, J)) break;
            const int fc0 = 2 * J;
            const int nnj = min(2, bv.nfrag - fc0);
            const int kend = min(8, 2 * (bv.nfrag - 4 * I));       // k-steps (4 rows of Dh each) in row block I
            // per-column constants of this thread's B fragments: column j = (fc0+nj)*8 + lr
            int sb[2], cbs[2], nB[2];
#pragma unroll
            for (int nj = 0; nj < 2; nj++) {
                const int j = (fc0 + nj) * 8 + lr;
                sb[nj] = nj < nnj ? s_colslot[j] : 255;
                cbs[nj] = sb[nj] != 255 ? s_colstart[sb[nj]] : 0;
                nB[nj] = sb[nj] != 255 ? s_colstart[sb[nj] + 1] - cbs[nj] : 0;
            }
            double acc[8][2][2];
#pragma unroll
            for (int mf = 0; mf < 8; mf++)
#pragma unroll
                for (int nj = 0; nj < 2; nj++) { acc[mf][nj][0] = 0.0; acc[mf][nj][1] = 0.0; }
            const double* pa = s_phi + (32 * I + lc) * LD + m0 * 8 + lr;
            for (int ks = 0; ks < kend; ks++) {
                const int i = 32 * I + 4 * ks + lc;
                const int sa = s_colslot[i];
                const int oa = sa != 255 ? i - s_colstart[sa] : 0;
                double bf[2];
#pragma unroll
                for (int nj = 0; nj < 2; nj++) {
                    double v = 0.0;
                    const int j = (fc0 + nj) * 8 + lr;
                    if (sb[nj] != 255 && (sa < sb[nj] || (sa == sb[nj] && i <= j))) {
                        const unsigned int off = s_boff[sa * g.max_nb + sb[nj]];
                        if (off != 0xffffffffu) v = __ldg(Dh + off + oa * nB[nj] + (j - cbs[nj]));
                    }
                    bf[nj] = v;
                }
                double a[8];
#pragma unroll
                for (int mf = 0; mf < 8; mf++) a[mf] = mf < nmf ? pa[4 * ks * LD + mf * 8] : 0.0;
#pragma unroll
                for (int mf = 0; mf < 8; mf++)
#pragma unroll
                    for (int nj = 0; nj < 2; nj++) dmma884(acc[mf][nj][0], acc[mf][nj][1], a[mf], bf[nj]);
            }
            // X[g][j] * Phi[g][j], g = (m0+mf)*8 + lr, j = (fc0+nj)*8 + 2*lc + e
#pragma unroll
            for (int nj = 0; nj < 2; nj++) {
                if (nj >= nnj) continue;
#pragma unroll
                for (int e = 0; e < 2; e++) {
                    const double* pj = s_phi + ((fc0 + nj) * 8 + 2 * lc + e) * LD + m0 * 8 + lr;
#pragma unroll
                    for (int mf = 0; mf < 8; mf++) if (mf < nmf) part[mf] = fma(acc[mf][nj][e], pj[mf * 8], part[mf]);
                }
            }
        }
#pragma unroll
        for (int mf = 0; mf < 8; mf++) {
            double v = part[mf];
            v += __shfl_xor_sync(0xffffffffu, v, 1);
            v += __shfl_xor_sync(0xffffffffu, v, 2);
            if (lc == 0 && mf < nmf) atomicAdd(&s_rho[(m0 + mf) * 8 + lr], v);
        }
    }
    __syncthreads();
    if ((int)threadIdx.x < bv.Kb) {
        const int q = threadIdx.x;
        int qk = q % bv.ez, qj = (q / bv.ez) % bv.ey, qi = q / (bv.ez * bv.ey);
        rho[((size_t)(bv.i0 + qi) * g.N[1] + (bv.j0 + qj)) * g.N[2] + (bv.k0 + qk)] = s_rho[q];
    }
}

// ---------------------------------------------------------------------------------------------------
// layout conversion (streaming, HBM-bound): public pair-list layout <-> canonical half
// One warp per public key: H_p = Hc_c (canonical key) or its transpose (mirror key).
__global__ void __launch_bounds__(256) k_expand_H(long long n_pairs, const long long* __restrict__ poff, const int* __restrict__ pcanon,
                                                  const unsigned char* __restrict__ pflag, const int* __restrict__ pnab,
                                                  const unsigned int* __restrict__ coff, const double* __restrict__ Hc, double* __restrict__ H) {
    const long long p = (long long)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (p >= n_pairs) return;
    const int lane = threadIdx.x & 31;
    const int nA = pnab[p] & 0xffff, nB = pnab[p] >> 16;
    const double* src = Hc + coff[pcanon[p]];
    double* dst = H + poff[p];
    if (pflag[p]) {
        for (int e = lane; e < nA * nB; e += 32) dst[e] = src[e];
    } else {                                            // canonical block is nB x nA; dst[i][j] = src[j][i]
        for (int e = lane; e < nA * nB; e += 32) { const int i = e / nB, j = e - i * nB; dst[e] = src[j * nA + i]; }
    }
}

// One warp per canonical key c = (A,B,n): Dh_c = D_(A,B,n) + D_(B,A,-n)^T; the on-site key (A,A,0) keeps
// D[i][i] on the diagonal, D[i][j] + D[j][i] above it and 0 below, so that the upper-triangle sum of k_rho
// reproduces the full ordered double sum of Eq. 3 without assuming any symmetry of D (reading R9).
__global__ void __launch_bounds__(256) k_sym_D(long long n_canon, const long long* __restrict__ poff, const int* __restrict__ cpub,
                                               const int* __restrict__ cmir, const int* __restrict__ pnab,
                                               const unsigned int* __restrict__ coff, const double* __restrict__ D, double* __restrict__ Dh) {
    const long long c = (long long)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (c >= n_canon) return;
    const int lane = threadIdx.x & 31;
    const int p = cpub[c], q = cmir[c];
    const int nA = pnab[p] & 0xffff, nB = pnab[p] >> 16;
    const double* d1 = D + poff[p];
    const double* d2 = D + poff[q];
    double* dst = Dh + coff[c];
    if (p == q) {
        for (int e = lane; e < nA * nB; e += 32) {
            const int i = e / nB, j = e - i * nB;
            dst[e] = i < j ? d1[e] + d1[j * nA + i] : (i == j ? d1[e] : 0.0);
        }
    } else {
        for (int e = lane; e < nA * nB; e += 32) { const int i = e / nB, j = e - i * nB; dst[e] = d1[e] + d2[j * nA + i]; }
    }
}

// ---------------------------------------------------------------------------------------------------
// algorithmic work counters (for the roofline numerator): per mesh point, the atoms with |d| < rc.
__global__ void __launch_bounds__(128) k_alg_stats(Geom g, long long n_batch, const int* __restrict__ order, const int* __restrict__ bstart,
                                                   const NeighEntry* __restrict__ bent, const double* __restrict__ atom_pos,
                                                   const int* __restrict__ atom_spec, const SpeciesDev* __restrict__ sp,
                                                   unsigned long long* __restrict__ out) {
    const int b = order[blockIdx.x];
    const int bz = b % g.nb[2], by = (b / g.nb[2]) % g.nb[1], bx = b / (g.nb[2] * g.nb[1]);
    const int i0 = bx * g.bs[0], j0 = by * g.bs[1], k0 = bz * g.bs[2];
    const int ey = min(g.bs[1], g.N[1] - j0), ez = min(g.bs[2], g.N[2] - k0);
    const int Kb = min(g.bs[0], g.N[0] - i0) * ey * ez;
    unsigned long long inc = 0, sn = 0, sn2 = 0, ne = 0;
    const int q = threadIdx.x;
    if (q < Kb) {
        double x, y, z;
        mesh_point(g, i0 + q / (ez * ey), j0 + (q / ez) % ey, k0 + q % ez, x, y, z);
        int na = 0, no = 0;
        for (int e = bstart[b]; e < bstart[b + 1]; e++) {
            const NeighEntry en = bent[e];
            int t1, t2, t3; unpack_shift(en.shift, t1, t2, t3);
            const double dx = x - (atom_pos[3 * en.atom + 0] + t1 * g.a[0] + t2 * g.a[3] + t3 * g.a[6]);
            const double dy = y - (atom_pos[3 * en.atom + 1] + t1 * g.a[1] + t2 * g.a[4] + t3 * g.a[7]);
            const double dz = z - (atom_pos[3 * en.atom + 2] + t1 * g.a[2] + t2 * g.a[5] + t3 * g.a[8]);
            const SpeciesDev* S = sp + atom_spec[en.atom];
            if (sqrt(dx * dx + dy * dy + dz * dz) < S->rc) { na++; no += S->norb; }
        }
        inc = na; sn = no; sn2 = (unsigned long long)no * no; ne = na > 0;
    }
    for (int d = 16; d; d >>= 1) {
        inc += __shfl_xor_sync(0xffffffffu, inc, d); sn += __shfl_xor_sync(0xffffffffu, sn, d);
        sn2 += __shfl_xor_sync(0xffffffffu, sn2, d); ne += __shfl_xor_sync(0xffffffffu, ne, d);
    }
    if ((threadIdx.x & 31) == 0) { atomicAdd(out + 0, inc); atomicAdd(out + 1, sn); atomicAdd(out + 2, sn2); atomicAdd(out + 3, ne); }
}

// ---------------------------------------------------------------------------------------------------
// host-side launchers
int gint_configure_kernels(gint_ctx* c) {
    const int smem = (int)c->smem_bytes;
    GINT_CUDA(cudaFuncSetAttribute(k_vlocal, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    GINT_CUDA(cudaFuncSetAttribute(k_rho, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    return GINT_OK;
}

int gint_launch_vlocal(gint_ctx* c, const double* V, double* H, cudaStream_t st) {
    GINT_CUDA(cudaSetDevice(c->device));
    if (c->n_values == 0) return GINT_OK;
    GINT_CUDA(cudaMemsetAsync(c->d_cval, 0, sizeof(double) * (size_t)c->n_cvalues, st));
    if (c->n_batch > 0) {
        GINT_CUDA(cudaEventRecord(c->ev[0], st));
        k_vlocal<<<(unsigned)c->n_batch, GINT_THREADS, c->smem_bytes, st>>>(c->geom, c->d_order, c->d_bstart, c->d_bent, c->d_atom_pos,
            c->d_atom_species, c->d_species, c->d_tab, c->d_crow, c->d_ckey, c->d_coff, V, c->d_cval);
        GINT_CUDA(cudaGetLastError());
        GINT_CUDA(cudaEventRecord(c->ev[1], st));
        c->timed[0] = true;
    }
    k_expand_H<<<(unsigned)((c->n_pairs + 7) / 8), 256, 0, st>>>(c->n_pairs, c->d_poff, c->d_pcanon, c->d_pflag, c->d_pnA, c->d_coff, c->d_cval, H);
    GINT_CUDA(cudaGetLastError());
    return GINT_OK;
}

int gint_launch_rho(gint_ctx* c, const double* D, double* rho, cudaStream_t st) {
    GINT_CUDA(cudaSetDevice(c->device));
    const size_t npts = (size_t)c->geom.N[0] * c->geom.N[1] * c->geom.N[2];
    GINT_CUDA(cudaMemsetAsync(rho, 0, sizeof(double) * npts, st));      // points of batches without neighbours
    if (c->n_batch == 0) return GINT_OK;
    k_sym_D<<<(unsigned)((c->n_canon + 7) / 8), 256, 0, st>>>(c->n_canon, c->d_poff, c->d_cpub, c->d_cmir, c->d_pnA, c->d_coff, D, c->d_cval);
    GINT_CUDA(cudaGetLastError());
    GINT_CUDA(cudaEventRecord(c->ev[2], st));
    k_rho<<<(unsigned)c->n_batch, GINT_THREADS, c->smem_bytes, st>>>(c->geom, c->d_order, c->d_bstart, c->d_bent, c->d_atom_pos,
        c->d_atom_species, c->d_species, c->d_tab, c->d_crow, c->d_ckey, c->d_coff, c->d_cval, rho);
    GINT_CUDA(cudaGetLastError());
    GINT_CUDA(cudaEventRecord(c->ev[3], st));
    c->timed[1] = true;
    return GINT_OK;
}

int gint_launch_alg_stats(gint_ctx* c) {
    GINT_CUDA(cudaSetDevice(c->device));
    unsigned long long* d_out;
    GINT_CUDA(cudaMalloc(&d_out, 4 * sizeof(unsigned long long)));
    GINT_CUDA(cudaMemset(d_out, 0, 4 * sizeof(unsigned long long)));
    if (c->n_batch > 0) {
        k_alg_stats<<<(unsigned)c->n_batch, GINT_MAX_K>>>(c->geom, c->n_batch, c->d_order, c->d_bstart, c->d_bent, c->d_atom_pos,
                                                          c->d_atom_species, c->d_species, d_out);
        GINT_CUDA(cudaGetLastError());
    }
    unsigned long long h[4];
    GINT_CUDA(cudaMemcpy(h, d_out, sizeof(h), cudaMemcpyDeviceToHost));
    GINT_CUDA(cudaFree(d_out));
    for (int i = 0; i < 4; i++) c->alg[i] = (long long)h[i];
    c->have_alg = true;
    return GINT_OK;
}
