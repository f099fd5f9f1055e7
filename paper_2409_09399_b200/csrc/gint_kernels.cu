// gint_kernels.cu -- the per-call hot path (north_star steps 2 and 3), fp64, sm_100a.
//
// Work decomposition.  The mesh is cut into grid batches (default 8x8x8 points) whose neighbouring
// atom images were listed by gint_init, most active first, and split into G groups of at most
// 8 atoms / 104 orbitals.  One CTA owns one TILE = (batch, group I, group J), I <= J: the 104 x 104 block of
// Phi_I^T diag(V dV) Phi_J (gint_vlocal, Eq. 2) or of the density blocks D_IJ (gint_rho, Eq. 3
// PAPER.md:73).  That block stays in REGISTERS (DMMA accumulators, resp. DMMA B fragments) while the CTA streams
// over the batch in chunks of 32 mesh points: all 16 warps first evaluate the orbitals of the <= 16 atoms of the
// tile at the chunk's points into shared memory (the paper's orbital-value kernel, never written to
// global memory), then contract them on the FP64 tensor pipe (mma.sync m8n8k4 f64 = DMMA.8x8x4).  Fragments
// (8 orbitals x 4 points) on which every atom is outside its cutoff sphere (Fig. 6: zero padding)
// are skipped with per-chunk bit masks, so zero padding costs (almost) no arithmetic.
// Only one of each mirror pair of blocks, (A,B,n) / (B,A,-n), is accumulated ("canonical half"); small
// streaming kernels convert between the public pair-list layout and the canonical layout.
#include "gint_internal.h"

// ---------------------------------------------------------------------------------------------------
// shared memory of the tile kernels
struct TileSmem {
    // phi[stage][side][orbital row][GINT_LD]: side 0 = group I, side 1 = group J (scaled by V dV in vlocal)
    double phi[2][2][GINT_TILE_ORB][GINT_LD];
    double pos[16][3];                  // slot s < 8: atom s of group I; slot 8 + s: atom s of group J
    double4 pts[2][GINT_CHUNK];         // [stage][point of the chunk]: x, y, z, weight (V dV in vlocal)
    double pvalid[2][GINT_CHUNK];       // 1 = the lane's point exists (inside the batch and the mesh), 0 = padding
    double red[GINT_CHUNK];             // rho: per-point partial sums of the chunk
    int spec[16];
    int atom[16];
    int shift[16];
    int cstart[2][GINT_TILE_ATOMS + 1]; // first orbital row of each atom inside its group
    unsigned int pair_off[GINT_TILE_ATOMS][GINT_TILE_ATOMS];   // canonical block offset of (I atom a, J atom b); ~0u = none
    unsigned char pair_tr[GINT_TILE_ATOMS][GINT_TILE_ATOMS];   // 1 = the canonical key is (b, a): transposed
    unsigned char row_atom[2][GINT_TILE_ORB];                  // orbital row -> atom slot inside the group (255 = padding)
    unsigned char row_orb[2][GINT_TILE_ORB];                   // orbital row -> orbital index inside the atom
    unsigned char frag_atoms[2][16];                           // fragment -> bit mask of the atoms it holds orbitals of
    unsigned char slot_mask[2][16];                            // [stage][slot]: bit k = atom active on k-step k of the chunk
};
size_t gint_smem_needed(const Geom&) { return sizeof(TileSmem); }

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}


// A predicated-off DMMA still occupies the FP64 tensor pipe for its full duration (measured), and ptxas turns
// `if (bit) dmma`, the arms of a C switch and short loops around a DMMA all into predicated DMMAs.  So the choice
// of which of a row's four column fragments to multiply is made by an indexed branch (brx.idx) written in PTX:
// sixteen entry points into chains of mma instructions, one per value of the 4-bit column mask.
#define GINT_MMA(c0, c1, a, b) "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {" c0 "," c1 "},{" a "},{" b "},{" c0 "," c1 "};\n\t"
// DMMA A x B_j into accumulator j for every set bit j of m (0..15); `A` and `B` are PTX operand names
#define GINT_MMA_CHAINS(D0, D1, D2, D3)                                                                       \
    "{\n\t"                                                                                                   \
    "ts: .branchtargets C0, C1, C2, C3, C4, C5, C6, C7, C8, C9, C10, C11, C12, C13, C14, C15;\n\t"              \
    "brx.idx %13, ts;\n\t"                                                                                    \
    "C15: " D0 "C14: " D1 "bra C12;\n\t"                                                                        \
    "C13: " D0 "C12: " D2 "C8: " D3 "bra C0;\n\t"                                                                \
    "C11: " D0 "C10: " D1 "bra C8;\n\t"                                                                         \
    "C9: " D0 "bra C8;\n\t"                                                                                    \
    "C7: " D0 "C6: " D1 "C4: " D2 "bra C0;\n\t"                                                                  \
    "C5: " D0 "bra C4;\n\t"                                                                                    \
    "C3: " D0 "C2: " D1 "bra C0;\n\t"                                                                           \
    "C1: " D0 "C0:\n\t"                                                                                        \
    "}"
// one k-step of one fragment row: acc[j] += a x b[j] for the set bits j of m
__device__ __forceinline__ void dmma_row(double (&acc)[4][2], double a, const double (&b)[4], unsigned m) {
    asm volatile(GINT_MMA_CHAINS(GINT_MMA("%0", "%1", "%8", "%9"), GINT_MMA("%2", "%3", "%8", "%10"),
                                 GINT_MMA("%4", "%5", "%8", "%11"), GINT_MMA("%6", "%7", "%8", "%12"))
                 : "+d"(acc[0][0]), "+d"(acc[0][1]), "+d"(acc[1][0]), "+d"(acc[1][1]), "+d"(acc[2][0]), "+d"(acc[2][1]),
                   "+d"(acc[3][0]), "+d"(acc[3][1])
                 : "d"(a), "d"(b[0]), "d"(b[1]), "d"(b[2]), "d"(b[3]), "r"(m));
}
// two k-steps (a0 x b0[j], a1 x b1[j]) into the same accumulators: the rho kernel's 8-orbital fragment row
__device__ __forceinline__ void dmma_row2(double (&acc)[4][2], double a0, double a1, const double (&b0)[4], const double (&b1)[4], unsigned m) {
    asm volatile(GINT_MMA_CHAINS(GINT_MMA("%0", "%1", "%8", "%9") GINT_MMA("%0", "%1", "%14", "%15"),
                                 GINT_MMA("%2", "%3", "%8", "%10") GINT_MMA("%2", "%3", "%14", "%16"),
                                 GINT_MMA("%4", "%5", "%8", "%11") GINT_MMA("%4", "%5", "%14", "%17"),
                                 GINT_MMA("%6", "%7", "%8", "%12") GINT_MMA("%6", "%7", "%14", "%18"))
                 : "+d"(acc[0][0]), "+d"(acc[0][1]), "+d"(acc[1][0]), "+d"(acc[1][1]), "+d"(acc[2][0]), "+d"(acc[2][1]),
                   "+d"(acc[3][0]), "+d"(acc[3][1])
                 : "d"(a0), "d"(b0[0]), "d"(b0[1]), "d"(b0[2]), "d"(b0[3]), "r"(m),
                   "d"(a1), "d"(b1[0]), "d"(b1[1]), "d"(b1[2]), "d"(b1[3]));
}

struct TileView {
    int b, I, J, G;                  // batch, groups
    int i0, j0, k0, ex, ey, ez;      // batch origin and extents (mesh points)
    int nkz, nks, nchunk;            // k-steps along z per column, k-steps of the batch, chunks of 8 k-steps
    int nI, nJ;                      // atoms in the two groups
    int nfI, nfJ;                    // fragments (8 orbitals) in the two groups
    bool diag;
};

// ---------------------------------------------------------------------------------------------------
// Tile set-up: atom slots, orbital-row maps, canonical block of every atom pair of the tile.
__device__ __forceinline__ void tile_setup(const Geom& g, TileSmem& S, TileView& tv, const int2* __restrict__ tile,
                                           const int* __restrict__ bstart, const NeighEntry* __restrict__ bent,
                                           const double* __restrict__ atom_pos, const int* __restrict__ atom_spec,
                                           const SpeciesDev* __restrict__ sp, const int* __restrict__ crow,
                                           const unsigned long long* __restrict__ ckey, const unsigned int* __restrict__ coff) {
    const int tid = threadIdx.x;
    const int2 td = tile[blockIdx.x];
    tv.b = td.x; tv.I = td.y & 255; tv.J = (td.y >> 8) & 255; tv.G = (td.y >> 16) & 255;
    tv.diag = tv.I == tv.J;
    const int b = tv.b;
    const int bz = b % g.nb[2], by = (b / g.nb[2]) % g.nb[1], bx = b / (g.nb[2] * g.nb[1]);
    tv.i0 = bx * g.bs[0]; tv.j0 = by * g.bs[1]; tv.k0 = bz * g.bs[2];
    tv.ex = min(g.bs[0], g.N[0] - tv.i0); tv.ey = min(g.bs[1], g.N[1] - tv.j0); tv.ez = min(g.bs[2], g.N[2] - tv.k0);
    tv.nkz = (tv.ez + 3) >> 2;
    tv.nks = tv.ex * tv.ey * tv.nkz;
    tv.nchunk = (tv.nks + 7) >> 3;
    const int e0 = bstart[b], n = bstart[b + 1] - e0;
    const int eI = group_begin(tv.I, n, tv.G), eJ = group_begin(tv.J, n, tv.G);
    tv.nI = group_begin(tv.I + 1, n, tv.G) - eI;
    tv.nJ = group_begin(tv.J + 1, n, tv.G) - eJ;

    if (tid < 16) {
        const int side = tid >> 3, a = tid & 7;
        const bool valid = a < (side ? tv.nJ : tv.nI);
        int atom = 0, shift = pack_shift(0, 0, 0), spec = 0;
        double x = 0, y = 0, z = 0;
        if (valid) {
            const NeighEntry e = bent[e0 + (side ? eJ : eI) + a];
            int t1, t2, t3; unpack_shift(e.shift, t1, t2, t3);
            atom = e.atom; shift = e.shift; spec = atom_spec[atom];
            x = atom_pos[3 * atom + 0] + t1 * g.a[0] + t2 * g.a[3] + t3 * g.a[6];
            y = atom_pos[3 * atom + 1] + t1 * g.a[1] + t2 * g.a[4] + t3 * g.a[7];
            z = atom_pos[3 * atom + 2] + t1 * g.a[2] + t2 * g.a[5] + t3 * g.a[8];
        }
        S.pos[tid][0] = x; S.pos[tid][1] = y; S.pos[tid][2] = z;
        S.spec[tid] = spec; S.atom[tid] = atom; S.shift[tid] = shift;
        S.slot_mask[0][tid] = 0; S.slot_mask[1][tid] = 0;
    }
    __syncthreads();
    if (tid < 2) {
        int o = 0;
        const int na = tid ? tv.nJ : tv.nI;
        for (int a = 0; a <= GINT_TILE_ATOMS; a++) { S.cstart[tid][a] = o; if (a < na) o += sp[S.spec[8 * tid + a]].norb; }
    }
    __syncthreads();
    const int totI = S.cstart[0][GINT_TILE_ATOMS], totJ = S.cstart[1][GINT_TILE_ATOMS];
    tv.nfI = (totI + 7) >> 3;
    tv.nfJ = (totJ + 7) >> 3;
    if (tid < 2 * GINT_TILE_ORB) {
        const int side = tid / GINT_TILE_ORB, row = tid - side * GINT_TILE_ORB;
        int a = 255, o = 0;
        for (int k = 0; k < GINT_TILE_ATOMS; k++)
            if (row >= S.cstart[side][k] && row < S.cstart[side][k + 1]) { a = k; o = row - S.cstart[side][k]; }
        S.row_atom[side][row] = (unsigned char)a; S.row_orb[side][row] = (unsigned char)o;
    } else if (tid < 2 * GINT_TILE_ORB + 32) {
        const int q = tid - 2 * GINT_TILE_ORB, side = q >> 4, f = q & 15;
        unsigned m = 0;
        for (int k = 0; k < GINT_TILE_ATOMS; k++)
            if (S.cstart[side][k] < 8 * f + 8 && S.cstart[side][k + 1] > 8 * f) m |= 1u << k;
        S.frag_atoms[side][f] = (unsigned char)m;
    } else if (tid >= 320 && tid < 320 + 64) {
        const int q = tid - 320, a = q >> 3, bb = q & 7;
        unsigned int off = 0xffffffffu; unsigned char tr = 0;
        // diagonal tile: only pairs a <= b are accumulated (a == b is the full on-site block)
        if (a < tv.nI && bb < tv.nJ && !(tv.diag && a > bb)) {
            int A = S.atom[a], B = S.atom[8 + bb];
            int ta1, ta2, ta3, tb1, tb2, tb3;
            unpack_shift(S.shift[a], ta1, ta2, ta3); unpack_shift(S.shift[8 + bb], tb1, tb2, tb3);
            int n1 = tb1 - ta1, n2 = tb2 - ta2, n3 = tb3 - ta3;
            const bool ge0 = n1 > 0 || (n1 == 0 && (n2 > 0 || (n2 == 0 && n3 >= 0)));
            if (!(A < B || (A == B && ge0))) { const int t = A; A = B; B = t; n1 = -n1; n2 = -n2; n3 = -n3; tr = 1; }
            const int m = g.key_m;
            if (abs(n1) <= m && abs(n2) <= m && abs(n3) <= m) {
                const unsigned long long M = (unsigned long long)g.key_M;
                const unsigned long long want = (((unsigned long long)B * M + (unsigned long long)(n1 + m)) * M + (unsigned long long)(n2 + m)) * M + (unsigned long long)(n3 + m);
                int lo = crow[A], hi = crow[A + 1] - 1;
                while (lo <= hi) {
                    const int mid = (lo + hi) >> 1;
                    const unsigned long long k = ckey[mid];
                    if (k == want) { off = coff[mid]; break; }
                    if (k < want) lo = mid + 1; else hi = mid - 1;
                }
            }
        }
        S.pair_off[a][bb] = off; S.pair_tr[a][bb] = tr;
    }
    // padding rows (orbital rows between the group's last orbital and the end of its last fragment) must hold zeros
    for (int idx = tid; idx < 2 * 2 * 8 * GINT_LD; idx += blockDim.x) {
        const int col = idx % GINT_LD, r = (idx / GINT_LD) & 7, side = (idx / (8 * GINT_LD)) & 1, st = idx / (16 * GINT_LD);
        const int row = (side ? totJ : totI) + r;
        if (row < GINT_TILE_ORB) S.phi[st][side][row][col] = 0.0;
    }
    __syncthreads();
}

// ---------------------------------------------------------------------------------------------------
// Orbital values of one atom at the 32 points of a chunk (north_star step 2): lane = point, the atom is
// warp-uniform.  phi = R_s(|d|) Y_lm(d/|d|), zero for |d| >= rc (Fig. 6); radial part:
// per-interval cubic in b = r/dr - i (reading R5).
//   mode 0: out0 <- phi            mode 1: out0 <- w phi
//   mode 2: out0 <- phi, out1 <- w phi          mode 3: out0 <- phi, out1 <- phi
// Returns the 8-bit k-step activity mask of the atom on this chunk (bit k: some point of k-step k is inside).
__device__ __forceinline__ unsigned eval_atom_chunk(const Geom& g, const SpeciesDev* __restrict__ S, const double* __restrict__ tab,
                                                   bool valid, double dx, double dy, double dz, int mode, double w,
                                                   double* __restrict__ out0, double* __restrict__ out1) {
    const int lane = threadIdx.x & 31;
    const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
    const double rc = S->rc;
    const bool inside = valid && r2 < rc * rc;
    const unsigned bal = __ballot_sync(0xffffffffu, inside);
    unsigned km = (bal | (bal >> 1) | (bal >> 2) | (bal >> 3)) & 0x11111111u;   // bit 4k = any of the 4 points of k-step k
    km = (km | (km >> 3)) & 0x03030303u; km = (km | (km >> 6)) & 0x000f000fu; km = (km | (km >> 12)) & 0xffu;
    const int norb = S->norb;
    double* o0 = out0 + lane;
    double* o1 = out1 + lane;
    if (bal == 0u) {
        for (int o = 0; o < norb; o++) { o0[o * GINT_LD] = 0.0; if (mode >= 2) o1[o * GINT_LD] = 0.0; }
        return 0u;
    }
    // lanes outside the sphere run the same instructions on a clamped radius and store zeros
    const double w0 = inside ? (mode == 1 ? w : 1.0) : 0.0;
    const double w1 = inside ? (mode == 2 ? w : 1.0) : 0.0;
    // 1/r by two Newton steps from the single-precision reciprocal square root (relative error ~1e-7 -> 1e-14 -> 1e-28)
    const double q = fmin(fmax(r2, 1e-30), rc * rc);
    double ir = (double)rsqrtf((float)q);
    ir = ir * fma(-0.5 * q, ir * ir, 1.5);
    ir = ir * fma(-0.5 * q, ir * ir, 1.5);
    const double r = q * ir;
    const int nsh = S->n_shell;
    const double x = r * g.inv_dr;
    int i = (int)x;
    i = min(i, S->n_int - 1);
    const double bq = x - (double)i;
    const double2* row = reinterpret_cast<const double2*>(tab) + ((size_t)S->tab_off + (size_t)i * nsh) * 2;
    const bool tiny = r < 1e-12;
    if (tiny) ir = 0.0;
    const double ux = dx * ir, uy = dy * ir, uz = dz * ir;
    const double lz = tiny ? 0.0 : 1.0;          // l > 0 orbitals vanish at the nucleus
    int o = 0;
#define GINT_PUT(v) do { const double v_ = (v); o0[o * GINT_LD] = w0 * v_; if (mode >= 2) o1[o * GINT_LD] = w1 * v_; o++; } while (0)
#pragma unroll 1
    for (int k = 0; k < nsh; k++) {
        const double2 c01 = __ldg(row + 2 * k), c23 = __ldg(row + 2 * k + 1);
        const double R = fma(fma(fma(c23.y, bq, c23.x), bq, c01.y), bq, c01.x);
        const int l = S->l[k];
        if (l == 0) {
            GINT_PUT(R * 0.28209479177387814);
        } else if (l == 1) {
            const double R1 = R * 0.4886025119029199;
            GINT_PUT(R1 * uy); GINT_PUT(R1 * uz); GINT_PUT(R1 * ux);
        } else {
            const double R2 = R * lz;
            const double c2 = R2 * 1.0925484305920792;
            GINT_PUT(c2 * ux * uy);
            GINT_PUT(c2 * uy * uz);
            GINT_PUT(R2 * 0.31539156525252005 * (3.0 * uz * uz - 1.0));
            GINT_PUT(c2 * ux * uz);
            GINT_PUT(R2 * 0.5462742152960396 * (ux * ux - uy * uy));
        }
    }
#undef GINT_PUT
    return km;
}

// mesh point of lane `lane` in chunk c of the batch: k-step ks = 8c + lane/4 = ((ix*ey)+iy)*nkz + kz, z = 4kz + lane%4
__device__ __forceinline__ bool chunk_point(const TileView& tv, int c, int lane, int& gi, int& gj, int& gk) {
    const int ks = 8 * c + (lane >> 2);
    const int kz = ks % tv.nkz, t = ks / tv.nkz;
    const int iy = t % tv.ey, ix = t / tv.ey;
    const int iz = 4 * kz + (lane & 3);
    gi = tv.i0 + ix; gj = tv.j0 + iy; gk = tv.k0 + iz;
    return ks < tv.nks && iz < tv.ez;
}

// Mesh points of chunk c (coordinates and the vlocal weight V dV) into pts[c & 1]; run by one warp, two chunks ahead
// of the evaluation that consumes them, so that the global load of V is off the critical path.
template <bool VLOCAL>
__device__ __forceinline__ void make_points(const Geom& g, TileSmem& S, const TileView& tv, int c, const double* __restrict__ V) {
    const int lane = threadIdx.x & 31;
    int gi, gj, gk;
    double4 p = make_double4(0.0, 0.0, 0.0, 0.0);
    double valid = 0.0;
    if (c < tv.nchunk && chunk_point(tv, c, lane, gi, gj, gk)) {
        mesh_point(g, gi, gj, gk, p.x, p.y, p.z);
        p.w = VLOCAL ? __ldg(V + ((size_t)gi * g.N[1] + gj) * g.N[2] + gk) * g.dV : 1.0;
        valid = 1.0;
    }
    S.pts[c & 1][lane] = p;
    S.pvalid[c & 1][lane] = valid;
}

// Evaluation phase of chunk c into pipeline stage st: warp w evaluates slot w (slot < 8: group I, else group J).
// vlocal: side I unscaled, side J scaled by V dV.  rho: both unscaled.  Diagonal tiles evaluate each atom once
// and write both sides.
template <bool VLOCAL>
__device__ __forceinline__ void eval_chunk(const Geom& g, TileSmem& S, const TileView& tv, int c, int st,
                                           const SpeciesDev* __restrict__ sp, const double* __restrict__ tab) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int side = warp >> 3, a = warp & 7;
    if (tv.diag ? (side == 1 || a >= tv.nI) : (a >= (side ? tv.nJ : tv.nI))) return;
    const double4 p = S.pts[st][lane];
    const bool valid = S.pvalid[st][lane] != 0.0;
    const SpeciesDev* Sp = sp + S.spec[warp];
    const double dx = p.x - S.pos[warp][0], dy = p.y - S.pos[warp][1], dz = p.z - S.pos[warp][2];
    double* out0 = &S.phi[st][side][S.cstart[side][a]][0];
    if (tv.diag) {
        double* out1 = &S.phi[st][1][S.cstart[0][a]][0];
        const unsigned km = eval_atom_chunk(g, Sp, tab, valid, dx, dy, dz, VLOCAL ? 2 : 3, p.w, out0, out1);
        if (lane == 0) { S.slot_mask[st][a] = (unsigned char)km; S.slot_mask[st][8 + a] = (unsigned char)km; }
    } else {
        const unsigned km = eval_atom_chunk(g, Sp, tab, valid, dx, dy, dz, (VLOCAL && side == 1) ? 1 : 0, p.w, out0, out0);
        if (lane == 0) S.slot_mask[st][warp] = (unsigned char)km;
    }
}

// rows / columns of the 4 x 4 warp grid: n fragments are dealt to 4 warps, the first (n % 4) get one more
__device__ __forceinline__ void warp_range(int n, int i, int& f0, int& nf) {
    const int base = n >> 2, rem = n & 3;
    f0 = i * base + min(i, rem); nf = base + (i < rem);
}
// 8-bit k-step mask of a fragment = OR of the masks of the atoms it holds orbitals of
__device__ __forceinline__ unsigned frag_kmask(const unsigned char* __restrict__ slot_mask8, unsigned atoms) {
    unsigned m = 0;
    while (atoms) { const int a = __ffs(atoms) - 1; atoms &= atoms - 1; m |= slot_mask8[a]; }
    return m;
}
// bit k of x -> bit 4k
__device__ __forceinline__ unsigned spread8(unsigned x) {
    x &= 0xffu; x = (x | (x << 12)) & 0x000f000fu; x = (x | (x << 6)) & 0x03030303u; x = (x | (x << 3)) & 0x11111111u;
    return x;
}
// Activity words of this warp's fragments on the chunk in stage st: nibble k of RW (CW) holds, for k-step k (FOLD:
// for the pair of k-steps 2k, 2k+1 = 8 points), one bit per fragment row (column) of the warp tile.
template <bool FOLD>
__device__ __forceinline__ void chunk_masks(const TileSmem& S, int st, int R0, int nr, int C0, int nc, unsigned& RW, unsigned& CW) {
    const int lane = threadIdx.x & 31;
    unsigned fm = 0;
    if (lane < 8) {
        const int side = lane >> 2, q = lane & 3;
        if (q < (side ? nc : nr)) {
            unsigned atoms = S.frag_atoms[side][(side ? C0 : R0) + q];
            while (atoms) { const int a = __ffs(atoms) - 1; atoms &= atoms - 1; fm |= S.slot_mask[st][8 * side + a]; }
        }
        if (FOLD) { fm = (fm | (fm >> 1)) & 0x55u; fm = (fm | (fm >> 1)) & 0x33u; fm = (fm | (fm >> 2)) & 0x0fu; }
        fm = spread8(fm) << q;
    }
    RW = __reduce_or_sync(0xffffffffu, lane < 4 ? fm : 0u);
    CW = __reduce_or_sync(0xffffffffu, lane >= 4 ? fm : 0u);
}
// fragment pairs this warp must compute: all of them, except, in a diagonal tile, those that hold no element with
// atom(row) <= atom(col)
__device__ __forceinline__ void warp_need(const TileSmem& S, const TileView& tv, int R0, int nr, int C0, int nc,
                                          unsigned ratoms[4], unsigned catoms[4], unsigned need[4]) {
#pragma unroll
    for (int i = 0; i < 4; i++) { ratoms[i] = i < nr ? S.frag_atoms[0][R0 + i] : 0u; catoms[i] = i < nc ? S.frag_atoms[1][C0 + i] : 0u; }
#pragma unroll
    for (int i = 0; i < 4; i++) {
        unsigned m = 0;
#pragma unroll
        for (int j = 0; j < 4; j++) {
            const bool nd = ratoms[i] && catoms[j] && (!tv.diag || (31 - __clz(catoms[j])) >= (__ffs(ratoms[i]) - 1));
            m |= nd ? 1u << j : 0u;
        }
        need[i] = m;
    }
}

// ---------------------------------------------------------------------------------------------------
// gint_vlocal main kernel (north_star step 3a): W_IJ = Phi_I^T diag(V dV) Phi_J accumulated over the whole batch in
// DMMA accumulators, then added to the canonical-half value array with fp64 reductions (red.global.add.f64):
// one reduction per element per batch.
__global__ void __launch_bounds__(GINT_THREADS, 1)
k_vlocal_tile(Geom g, const int2* __restrict__ tile, const int* __restrict__ bstart, const NeighEntry* __restrict__ bent,
              const double* __restrict__ atom_pos, const int* __restrict__ atom_spec, const SpeciesDev* __restrict__ sp,
              const double* __restrict__ tab, const int* __restrict__ crow, const unsigned long long* __restrict__ ckey,
              const unsigned int* __restrict__ coff, const double* __restrict__ V, double* __restrict__ Hc) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TileSmem& S = *reinterpret_cast<TileSmem*>(smem_raw);
    TileView tv;
    tile_setup(g, S, tv, tile, bstart, bent, atom_pos, atom_spec, sp, crow, ckey, coff);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, lr = lane >> 2, lc = lane & 3;
    // warp (wr, wc) of the 4 x 4 grid; the warps of one scheduler (warp % 4) sit on a diagonal so that the
    // schedulers get equal numbers of fragments although 13 = 4 + 3 + 3 + 3
    const int wr = warp >> 2, wc = ((warp & 3) + wr) & 3;
    int R0, nr, C0, nc;
    warp_range(tv.nfI, wr, R0, nr);
    warp_range(tv.nfJ, wc, C0, nc);
    unsigned ratoms[4], catoms[4], need[4];
    warp_need(S, tv, R0, nr, C0, nc, ratoms, catoms, need);
    double acc[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 4; j++) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }

    if (warp < 2) make_points<true>(g, S, tv, warp, V);
    __syncthreads();
    eval_chunk<true>(g, S, tv, 0, 0, sp, tab);
    for (int c = 0; c < tv.nchunk; c++) {
        const int st = c & 1;
        __syncthreads();                       // stage st is complete; every warp has finished the MMAs of chunk c-1
        if (warp == ((c + 2) & 15)) make_points<true>(g, S, tv, c + 2, V);
        if (c + 1 < tv.nchunk) eval_chunk<true>(g, S, tv, c + 1, st ^ 1, sp, tab);
        unsigned RW, CW;
        chunk_masks<false>(S, st, R0, nr, C0, nc, RW, CW);
        unsigned act = (RW | (RW >> 1) | (RW >> 2) | (RW >> 3)) & (CW | (CW >> 1) | (CW >> 2) | (CW >> 3)) & 0x11111111u;
        const double* pa = &S.phi[st][0][R0 * 8 + lr][lc];
        const double* pb = &S.phi[st][1][C0 * 8 + lr][lc];
        while (act) {
            const int p4 = __ffs(act) - 1; act &= act - 1;           // p4 = 4 * k-step
            const unsigned r4 = RW >> p4, c4 = (CW >> p4) & 15u;
            double bf[4];
#pragma unroll
            for (int j = 0; j < 4; j++) bf[j] = pb[j * 8 * GINT_LD + p4];      // inactive fragments: loaded, never used
#pragma unroll
            for (int i = 0; i < 4; i++) {
                if (!((r4 >> i) & 1u)) continue;
                const double a = pa[i * 8 * GINT_LD + p4];
                dmma_row(acc[i], a, bf, c4 & need[i]);
            }
        }
    }
    // flush: element (row, col) -> atom pair (a, b), orbitals (oa, ob) -> canonical block, transposed if the canonical
    // key is (b, a).  Exact zeros (fragments never touched, atoms that do not overlap inside this batch) are skipped.
#pragma unroll
    for (int i = 0; i < 4; i++) {
#pragma unroll
        for (int j = 0; j < 4; j++) {
            if (!((need[i] >> j) & 1u)) continue;
            const int row = (R0 + i) * 8 + lr;
            const int a = S.row_atom[0][row], oa = S.row_orb[0][row];
            if (a == 255) continue;
#pragma unroll
            for (int e = 0; e < 2; e++) {
                const double v = acc[i][j][e];
                const int col = (C0 + j) * 8 + 2 * lc + e;
                const int bb = S.row_atom[1][col], ob = S.row_orb[1][col];
                if (bb == 255 || v == 0.0) continue;
                const unsigned off = S.pair_off[a][bb];
                if (off == 0xffffffffu) continue;
                const int nA = S.cstart[0][a + 1] - S.cstart[0][a], nB = S.cstart[1][bb + 1] - S.cstart[1][bb];
                atomicAdd(Hc + off + (S.pair_tr[a][bb] ? ob * nA + oa : oa * nB + ob), v);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// gint_rho main kernel (north_star step 3b): the density blocks Dh_IJ of the tile are the stationary DMMA B
// fragments (registers); per chunk X = Phi_I Dh_IJ (32 points x 104) and rho_g += sum_j X_gj Phi_J,gj.
// Dh = canonical-half, symmetrised density blocks (k_sym_D).  Warp (wr, wc): rows (k) and columns (n) of Dh.
__device__ __forceinline__ unsigned fold_pairs(unsigned m) {     // 8 k-step bits -> 4 bits, one per 8 points
    m = (m | (m >> 1)) & 0x55u; m = (m | (m >> 1)) & 0x33u; m = (m | (m >> 2)) & 0x0fu;
    return m;
}
__global__ void __launch_bounds__(GINT_THREADS, 1)
k_rho_tile(Geom g, const int2* __restrict__ tile, const int* __restrict__ bstart, const NeighEntry* __restrict__ bent,
           const double* __restrict__ atom_pos, const int* __restrict__ atom_spec, const SpeciesDev* __restrict__ sp,
           const double* __restrict__ tab, const int* __restrict__ crow, const unsigned long long* __restrict__ ckey,
           const unsigned int* __restrict__ coff, const double* __restrict__ Dh, double* __restrict__ rho) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TileSmem& S = *reinterpret_cast<TileSmem*>(smem_raw);
    TileView tv;
    tile_setup(g, S, tv, tile, bstart, bent, atom_pos, atom_spec, sp, crow, ckey, coff);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, lr = lane >> 2, lc = lane & 3;
    const int wr = warp >> 2, wc = ((warp & 3) + wr) & 3;
    int R0, nr, C0, nc;
    warp_range(tv.nfI, wr, R0, nr);       // rows of Dh (orbitals of group I), 8 per fragment = 2 DMMA k-steps
    warp_range(tv.nfJ, wc, C0, nc);       // columns of Dh (orbitals of group J)
    unsigned ratoms[4], catoms[4], need[4];
    warp_need(S, tv, R0, nr, C0, nc, ratoms, catoms, need);
    // stationary B fragments: dreg[i][h][j] = Dh[row (R0+i)*8 + 4h + lc][col (C0+j)*8 + lr]
    double dreg[4][2][4];
#pragma unroll
    for (int i = 0; i < 4; i++)
#pragma unroll
        for (int h = 0; h < 2; h++)
#pragma unroll
            for (int j = 0; j < 4; j++) {
                double v = 0.0;
                if ((need[i] >> j) & 1u) {
                    const int row = (R0 + i) * 8 + 4 * h + lc, col = (C0 + j) * 8 + lr;
                    const int a = S.row_atom[0][row], bb = S.row_atom[1][col];
                    if (a != 255 && bb != 255) {
                        const unsigned off = S.pair_off[a][bb];
                        if (off != 0xffffffffu) {
                            const int oa = S.row_orb[0][row], ob = S.row_orb[1][col];
                            const int nA = S.cstart[0][a + 1] - S.cstart[0][a], nB = S.cstart[1][bb + 1] - S.cstart[1][bb];
                            v = __ldg(Dh + off + (S.pair_tr[a][bb] ? ob * nA + oa : oa * nB + ob));
                        }
                    }
                }
                dreg[i][h][j] = v;
            }

    if (warp < 2) make_points<false>(g, S, tv, warp, nullptr);
    __syncthreads();
    eval_chunk<false>(g, S, tv, 0, 0, sp, tab);
    for (int c = 0; c < tv.nchunk; c++) {
        const int st = c & 1;
        if (threadIdx.x < GINT_CHUNK) S.red[threadIdx.x] = 0.0;
        __syncthreads();
        if (warp == ((c + 2) & 15)) make_points<false>(g, S, tv, c + 2, nullptr);
        if (c + 1 < tv.nchunk) eval_chunk<false>(g, S, tv, c + 1, st ^ 1, sp, tab);
        unsigned RW, CW;                        // nibble pf: fragments active on the 8 points 8pf .. 8pf+7
        chunk_masks<true>(S, st, R0, nr, C0, nc, RW, CW);
        unsigned act = (RW | (RW >> 1) | (RW >> 2) | (RW >> 3)) & (CW | (CW >> 1) | (CW >> 2) | (CW >> 3)) & 0x1111u;
        while (act) {
            const int p4 = __ffs(act) - 1; act &= act - 1;
            const int pf = p4 >> 2;
            const unsigned r4 = (RW >> p4) & 15u, c4 = (CW >> p4) & 15u;
            double x[4][2];
#pragma unroll
            for (int j = 0; j < 4; j++) { x[j][0] = 0.0; x[j][1] = 0.0; }
            // A fragment: Phi_I[point 8pf + lr][orbital row (R0+i)*8 + 4h + lc]
            const double* pa = &S.phi[st][0][R0 * 8 + lc][8 * pf + lr];
#pragma unroll
            for (int i = 0; i < 4; i++) {
                const unsigned m = ((r4 >> i) & 1u) ? (c4 & need[i]) : 0u;
                if (!m) continue;
                const double a0 = pa[(i * 8) * GINT_LD], a1 = pa[(i * 8 + 4) * GINT_LD];
                dmma_row2(x, a0, a1, dreg[i][0], dreg[i][1], m);
            }
            // rho partial of point 8pf + lr: sum over this warp's columns of X * Phi_J
            double part = 0.0;
            const double* pj = &S.phi[st][1][C0 * 8 + 2 * lc][8 * pf + lr];
#pragma unroll
            for (int j = 0; j < 4; j++) {
                if (!((c4 >> j) & 1u)) continue;
                part = fma(x[j][0], pj[(j * 8) * GINT_LD], part);
                part = fma(x[j][1], pj[(j * 8 + 1) * GINT_LD], part);
            }
            part += __shfl_xor_sync(0xffffffffu, part, 1);
            part += __shfl_xor_sync(0xffffffffu, part, 2);
            if (lc == 0 && part != 0.0) atomicAdd(&S.red[8 * pf + lr], part);
        }
        __syncthreads();
        if (threadIdx.x < GINT_CHUNK) {
            const double v = S.red[threadIdx.x];
            int gi, gj, gk;
            if (v != 0.0 && chunk_point(tv, c, threadIdx.x, gi, gj, gk))
                atomicAdd(rho + ((size_t)gi * g.N[1] + gj) * g.N[2] + gk, v);
        }
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

// One warp per canonical key c = (A,B,n): Dh_c = D_(A,B,n) + D_(B,A,-n)^T; the self key (A,A,0) keeps
// D[i][i] on the diagonal, D[i][j] + D[j][i] above it and 0 below, so that summing every unordered pair of atom
// images once reproduces the full ordered double sum of Eq. 3 without assuming any symmetry of D (reading R9).
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
__global__ void __launch_bounds__(128) k_alg_stats(Geom g, const int* __restrict__ bstart,
                                                   const NeighEntry* __restrict__ bent, const double* __restrict__ atom_pos,
                                                   const int* __restrict__ atom_spec, const SpeciesDev* __restrict__ sp,
                                                   unsigned long long* __restrict__ out) {
    const int b = blockIdx.x;
    const int bz = b % g.nb[2], by = (b / g.nb[2]) % g.nb[1], bx = b / (g.nb[2] * g.nb[1]);
    const int i0 = bx * g.bs[0], j0 = by * g.bs[1], k0 = bz * g.bs[2];
    const int ey = min(g.bs[1], g.N[1] - j0), ez = min(g.bs[2], g.N[2] - k0);
    const int Kb = min(g.bs[0], g.N[0] - i0) * ey * ez;
    unsigned long long inc = 0, sn = 0, sn2 = 0, ne = 0;
    if (bstart[b + 1] > bstart[b]) {
        for (int q = threadIdx.x; q < Kb; q += blockDim.x) {
            double x, y, z;
            mesh_point(g, i0 + q / (ez * ey), j0 + (q / ez) % ey, k0 + q % ez, x, y, z);
            int na = 0, no = 0;
            for (int e = bstart[b]; e < bstart[b + 1]; e++) {
                const NeighEntry en = bent[e];
                int t1, t2, t3; unpack_shift(en.shift, t1, t2, t3);
                const double dx = x - (atom_pos[3 * en.atom + 0] + t1 * g.a[0] + t2 * g.a[3] + t3 * g.a[6]);
                const double dy = y - (atom_pos[3 * en.atom + 1] + t1 * g.a[1] + t2 * g.a[4] + t3 * g.a[7]);
                const double dz = z - (atom_pos[3 * en.atom + 2] + t1 * g.a[2] + t2 * g.a[5] + t3 * g.a[8]);
                const SpeciesDev* Sp = sp + atom_spec[en.atom];
                if (sqrt(dx * dx + dy * dy + dz * dz) < Sp->rc) { na++; no += Sp->norb; }
            }
            inc += na; sn += no; sn2 += (unsigned long long)no * no; ne += na > 0;
        }
    }
    for (int d = 16; d; d >>= 1) {
        inc += __shfl_xor_sync(0xffffffffu, inc, d); sn += __shfl_xor_sync(0xffffffffu, sn, d);
        sn2 += __shfl_xor_sync(0xffffffffu, sn2, d); ne += __shfl_xor_sync(0xffffffffu, ne, d);
    }
    if ((threadIdx.x & 31) == 0 && inc) { atomicAdd(out + 0, inc); atomicAdd(out + 1, sn); atomicAdd(out + 2, sn2); atomicAdd(out + 3, ne); }
}

// ---------------------------------------------------------------------------------------------------
// host-side launchers
int gint_configure_kernels(gint_ctx* c) {
    const int smem = (int)c->smem_bytes;
    GINT_CUDA(cudaFuncSetAttribute(k_vlocal_tile, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    GINT_CUDA(cudaFuncSetAttribute(k_rho_tile, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    return GINT_OK;
}

int gint_launch_vlocal(gint_ctx* c, const double* V, double* H, cudaStream_t st) {
    GINT_CUDA(cudaSetDevice(c->device));
    if (c->n_values == 0) return GINT_OK;
    GINT_CUDA(cudaMemsetAsync(c->d_cval, 0, sizeof(double) * (size_t)c->n_cvalues, st));
    if (c->n_tiles > 0) {
        GINT_CUDA(cudaEventRecord(c->ev[0], st));
        k_vlocal_tile<<<(unsigned)c->n_tiles, GINT_THREADS, c->smem_bytes, st>>>(c->geom, c->d_tile, c->d_bstart, c->d_bent, c->d_atom_pos,
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
    GINT_CUDA(cudaMemsetAsync(rho, 0, sizeof(double) * npts, st));
    if (c->n_tiles == 0) return GINT_OK;
    k_sym_D<<<(unsigned)((c->n_canon + 7) / 8), 256, 0, st>>>(c->n_canon, c->d_poff, c->d_cpub, c->d_cmir, c->d_pnA, c->d_coff, D, c->d_cval);
    GINT_CUDA(cudaGetLastError());
    GINT_CUDA(cudaEventRecord(c->ev[2], st));
    k_rho_tile<<<(unsigned)c->n_tiles, GINT_THREADS, c->smem_bytes, st>>>(c->geom, c->d_tile, c->d_bstart, c->d_bent, c->d_atom_pos,
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
    if (c->n_batch_total > 0) {
        k_alg_stats<<<(unsigned)c->n_batch_total, 128>>>(c->geom, c->d_bstart, c->d_bent, c->d_atom_pos, c->d_atom_species, c->d_species, d_out);
        GINT_CUDA(cudaGetLastError());
    }
    unsigned long long h[4];
    GINT_CUDA(cudaMemcpy(h, d_out, sizeof(h), cudaMemcpyDeviceToHost));
    GINT_CUDA(cudaFree(d_out));
    for (int i = 0; i < 4; i++) c->alg[i] = (long long)h[i];
    c->have_alg = true;
    return GINT_OK;
}
