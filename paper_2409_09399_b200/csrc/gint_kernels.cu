// gint_kernels.cu -- the per-call hot path (north_star steps 2 and 3), fp64, sm_100a.
//
// Work decomposition.  The mesh is cut into grid batches (default 8x8x8 points) whose neighbouring
// atom images were listed by gint_init, most active first, each with a 64-bit ACTIVITY MASK over the
// batch's 4x4x4 "cubelets" of 2x2x2 mesh points (bit set = some point of the cubelet lies inside the atom's cutoff
// sphere; Fig. 6: everything else is zero padding).  The neighbours of a batch are split into G
// groups of at most 8 atoms / 104 orbitals.  One CTA owns one TILE = (batch, group I, group J), I <= J: the
// 104 x 104 block of Phi_I^T diag(V dV) Phi_J (gint_vlocal, Eq. 2) or of the density blocks D_IJ
// (gint_rho, Eq. 3).  That block stays in REGISTERS (DMMA accumulators, resp. stationary DMMA
// operands): the 13 x 13 fragments (8 x 8 orbitals) of the block are cut into SEGMENTS of one row fragment x up to
// 7 column fragments, four segments per consumer warp, dealt to the 8 consumer warps so that the four SM sub-partitions carry equal
// numbers of DMMAs; in a diagonal tile (I == J) only the fragments on or above the atom diagonal are segments.
// The CTA walks over the cubelets on which both groups are active, 4 cubelets (32 points) per pipeline stage: the
// orbital values of the needed (atom, cubelet) items are evaluated into shared memory (the paper's orbital-value
// kernel, never written to global memory; items compacted so that a quarter warp = one atom on one
// cubelet), then every warp runs the DMMA chains (mma.sync m8n8k4 f64 = DMMA.8x8x4) of its segments on the cubelets
// where the segment is active -- straight-line code specialised on the segment length, one bit test per cubelet.
// Only one of each mirror pair of blocks, (A,B,n) / (B,A,-n), is accumulated ("canonical half"); small
// streaming kernels convert between the public pair-list layout and the canonical layout.
#include "gint_internal.h"

typedef unsigned long long u64;
#define GINT_EVAL_GROUP 3          // radial shells whose spline coefficients are loaded together (registers vs memory-level parallelism)

// ---------------------------------------------------------------------------------------------------
// shared memory of the tile kernels
struct PairEnt { unsigned off; unsigned short sr, sc; };   // element (oa, ob) of the atom pair at off + oa*sr + ob*sc; off = ~0u: none
struct SlotInfo { double rc2; int n_int, nsh, tab_off, lpack; };   // lpack: 2 bits of l per shell

struct TileView {
    int b, I, J, G;                  // batch, groups
    int i0, j0, k0, ex, ey, ez;      // batch origin and extents (mesh points)
    int nchunk;                      // stages of 4 cubelets
    int nI, nJ;                      // atoms in the two groups
    int nfI, nfJ;                    // fragments (8 orbitals) in the two groups
    bool diag;
};

struct TileSmem {
    // phi[stage][side][orbital row][GINT_LD]: side 0 = group I, side 1 = group J (scaled by V dV in vlocal);
    // column 8q + p = point p of the stage's q-th cubelet
    double phi[GINT_STAGES][2][GINT_TILE_ORB][GINT_LD];
    double4 pts[2][GINT_CHUNK];         // [stage][point]: x, y, z, weight (V dV in vlocal, 1 in rho)
    u64 full[GINT_STAGES], empty[GINT_STAGES];   // mbarriers: stage written by all producer warps / read by all consumer warps
    double pos[16][4];                  // slot s < 8: atom s of group I; slot 8 + s: atom s of group J
    SlotInfo sinfo[16];
    u64 amask[16];                      // cubelets on which the slot's atom is non-zero
    u64 need[16];                       // cubelets on which the slot's orbital rows are read by some segment
    u64 fmask[2][16];                   // [side][fragment]: OR of amask over the atoms with orbitals in the fragment
    u64 hmask[2];                       // side J: OR of fmask over the column fragments 0..6 / 7..12
    u64 U;                              // cubelets the tile walks over: (any I fragment) & (any J fragment)
    PairEnt pair[GINT_TILE_ATOMS][GINT_TILE_ATOMS];   // canonical block of (I atom a, J atom b)
    int atom[16], shift[16], spec[16];
    int cstart[2][GINT_TILE_ATOMS + 1]; // first orbital row of each atom inside its group
    int seg[GINT_MAX_SEG];              // slot (consumer warp) + 8 k: row fragment | first column fragment << 8 | n columns << 16
    int nitem[2], neval[2];             // [stage]: items of the stage, of which the first neval need a real evaluation
    int ncub;
    TileView tv;                        // written by tile_setup; read from here afterwards to keep registers free
    unsigned char valid[2][GINT_CHUNK]; // the stage's point exists (inside the batch and the mesh)
    unsigned char item[2][64];          // [stage][k]: slot << 2 | cubelet of the stage
    unsigned char cub[64 + 4];          // the tile's cubelets (bit numbers of U, ascending)
    unsigned char row_atom[2][GINT_TILE_ORB];   // orbital row -> atom slot inside the group (255 = padding)
    unsigned char row_orb[2][GINT_TILE_ORB];    // orbital row -> orbital index inside the atom
    unsigned char frag_atoms[2][16];            // fragment -> bit mask of the atoms it holds orbitals of
};
size_t gint_smem_needed(const Geom&) { return sizeof(TileSmem); }

// The DMMA chains and their operand loads are volatile asm: left to itself the compiler sinks every shared load to
// just before its DMMA (one operand register, fully serialised LDS -> DMMA -> LDS ...) and pairs the two k-steps of
// an accumulator back to back.  Volatile asm keeps the written order: all loads of a cubelet, then the DMMAs.
__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};" : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}
__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ double2 lds128(unsigned addr) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ double lds64(unsigned addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr) : "memory");
    return v;
}


__device__ __forceinline__ void mbar_init(u64* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ u64 warp_or64(u64 v) {
    const unsigned lo = __reduce_or_sync(0xffffffffu, (unsigned)v), hi = __reduce_or_sync(0xffffffffu, (unsigned)(v >> 32));
    return (u64)lo | ((u64)hi << 32);
}
__device__ __forceinline__ u64 shfl64(u64 v, int src) {
    const unsigned lo = __shfl_sync(0xffffffffu, (unsigned)v, src), hi = __shfl_sync(0xffffffffu, (unsigned)(v >> 32), src);
    return (u64)lo | ((u64)hi << 32);
}

// ---------------------------------------------------------------------------------------------------
// Tile set-up: atom slots, orbital-row maps, canonical block of every atom pair of the tile, activity masks,
// cubelet list, segments.
__device__ __forceinline__ void tile_setup(const Geom& g, TileSmem& S, TileView& tv, const int2* __restrict__ tile,
                                           const int* __restrict__ bstart, const NeighEntry* __restrict__ bent,
                                           const double* __restrict__ atom_pos, const int* __restrict__ atom_spec,
                                           const SpeciesDev* __restrict__ sp, const int* __restrict__ crow,
                                           const u64* __restrict__ ckey, const unsigned int* __restrict__ coff) {
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int2 td = tile[blockIdx.x];
    tv.b = td.x; tv.I = td.y & 255; tv.J = (td.y >> 8) & 255; tv.G = (td.y >> 16) & 255;
    tv.diag = tv.I == tv.J;
    const int b = tv.b;
    const int bz = b % g.nb[2], by = (b / g.nb[2]) % g.nb[1], bx = b / (g.nb[2] * g.nb[1]);
    tv.i0 = bx * g.bs[0]; tv.j0 = by * g.bs[1]; tv.k0 = bz * g.bs[2];
    tv.ex = min(g.bs[0], g.N[0] - tv.i0); tv.ey = min(g.bs[1], g.N[1] - tv.j0); tv.ez = min(g.bs[2], g.N[2] - tv.k0);
    const int e0 = bstart[b], n = bstart[b + 1] - e0;
    const int eI = group_begin(tv.I, n, tv.G), eJ = group_begin(tv.J, n, tv.G);
    tv.nI = group_begin(tv.I + 1, n, tv.G) - eI;
    tv.nJ = group_begin(tv.J + 1, n, tv.G) - eJ;

    if (tid < 16) {
        const int side = tid >> 3, a = tid & 7;
        const bool valid = a < (side ? tv.nJ : tv.nI);
        int atom = 0, shift = pack_shift(0, 0, 0), spec = 0;
        double x = 0, y = 0, z = 0;
        u64 m = 0;
        if (valid) {
            const NeighEntry e = bent[e0 + (side ? eJ : eI) + a];
            int t1, t2, t3; unpack_shift(e.shift, t1, t2, t3);
            atom = e.atom; shift = e.shift; spec = atom_spec[atom]; m = e.mask;
            x = atom_pos[3 * atom + 0] + t1 * g.a[0] + t2 * g.a[3] + t3 * g.a[6];
            y = atom_pos[3 * atom + 1] + t1 * g.a[1] + t2 * g.a[4] + t3 * g.a[7];
            z = atom_pos[3 * atom + 2] + t1 * g.a[2] + t2 * g.a[5] + t3 * g.a[8];
        }
        S.pos[tid][0] = x; S.pos[tid][1] = y; S.pos[tid][2] = z; S.pos[tid][3] = 0.0;
        S.spec[tid] = spec; S.atom[tid] = atom; S.shift[tid] = shift; S.amask[tid] = m;
        const SpeciesDev* Sp = sp + spec;
        SlotInfo si; si.rc2 = Sp->rc * Sp->rc; si.n_int = Sp->n_int; si.nsh = valid ? Sp->n_shell : 0; si.tab_off = Sp->tab_off;
        int lp = 0;
        for (int k = 0; k < Sp->n_shell; k++) lp |= Sp->l[k] << (2 * k);
        si.lpack = lp;
        S.sinfo[tid] = si;
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
        u64 fm = 0;
        for (int k = 0; k < GINT_TILE_ATOMS; k++)
            if (S.cstart[side][k] < 8 * f + 8 && S.cstart[side][k + 1] > 8 * f) { m |= 1u << k; fm |= S.amask[8 * side + k]; }
        S.frag_atoms[side][f] = (unsigned char)m;
        S.fmask[side][f] = fm;
    } else if (tid >= 256 && tid < 256 + 64) {
        const int q = tid - 256, a = q >> 3, bb = q & 7;
        PairEnt pe; pe.off = 0xffffffffu; pe.sr = 0; pe.sc = 0;
        // diagonal tile: only pairs a <= b are accumulated (a == b is the full on-site block)
        if (a < tv.nI && bb < tv.nJ && !(tv.diag && a > bb)) {
            int A = S.atom[a], B = S.atom[8 + bb];
            const int nA = S.cstart[0][a + 1] - S.cstart[0][a], nB = S.cstart[1][bb + 1] - S.cstart[1][bb];
            int ta1, ta2, ta3, tb1, tb2, tb3;
            unpack_shift(S.shift[a], ta1, ta2, ta3); unpack_shift(S.shift[8 + bb], tb1, tb2, tb3);
            int n1 = tb1 - ta1, n2 = tb2 - ta2, n3 = tb3 - ta3;
            const bool ge0 = n1 > 0 || (n1 == 0 && (n2 > 0 || (n2 == 0 && n3 >= 0)));
            bool tr = false;
            if (!(A < B || (A == B && ge0))) { const int t = A; A = B; B = t; n1 = -n1; n2 = -n2; n3 = -n3; tr = true; }
            const int m = g.key_m;
            if (abs(n1) <= m && abs(n2) <= m && abs(n3) <= m) {
                const u64 M = (u64)g.key_M;
                const u64 want = (((u64)B * M + (u64)(n1 + m)) * M + (u64)(n2 + m)) * M + (u64)(n3 + m);
                int lo = crow[A], hi = crow[A + 1] - 1;
                while (lo <= hi) {
                    const int mid = (lo + hi) >> 1;
                    const u64 k = ckey[mid];
                    if (k == want) { pe.off = coff[mid]; break; }
                    if (k < want) lo = mid + 1; else hi = mid - 1;
                }
            }
            // canonical key (b, a): the stored block is nB x nA and holds the transpose
            pe.sr = (unsigned short)(tr ? 1 : nB); pe.sc = (unsigned short)(tr ? nA : 1);
        }
        S.pair[a][bb] = pe;
    }
    // padding rows (orbital rows between the group's last orbital and the end of its last fragment) must hold zeros
    for (int idx = tid; idx < GINT_STAGES * 2 * 8 * GINT_LD; idx += blockDim.x) {
        const int col = idx % GINT_LD, r = (idx / GINT_LD) & 7, side = (idx / (8 * GINT_LD)) & 1, st = idx / (16 * GINT_LD);
        const int row = (side ? totJ : totI) + r;
        if (row < GINT_TILE_ORB) S.phi[st][side][row][col] = 0.0;
    }
    __syncthreads();
    if (warp == 0) {
        // union masks, cubelet list, per-slot read sets
        const u64 vI = lane < tv.nfI ? S.fmask[0][lane] : 0ull;
        const u64 vJ = lane < tv.nfJ ? S.fmask[1][lane] : 0ull;
        const u64 anyI = warp_or64(vI);
        const u64 h0 = warp_or64(lane < GINT_SEG_COLS ? vJ : 0ull) & anyI, h1 = warp_or64(lane >= GINT_SEG_COLS ? vJ : 0ull) & anyI;
        const u64 U = h0 | h1;
        const unsigned Ulo = (unsigned)U, Uhi = (unsigned)(U >> 32), lt = (1u << lane) - 1u;
        if ((Ulo >> lane) & 1u) S.cub[__popc(Ulo & lt)] = (unsigned char)lane;
        if ((Uhi >> lane) & 1u) S.cub[__popc(Ulo) + __popc(Uhi & lt)] = (unsigned char)(32 + lane);
        const int ncub = __popc(Ulo) + __popc(Uhi);
        if (lane < 4) S.cub[ncub + lane] = 0;
        u64 m = 0;
        if (lane < 16) {
            const int side = lane >> 3, a = lane & 7;
            const int nf = side ? tv.nfJ : tv.nfI;
            for (int f = 0; f < nf; f++)
                if ((S.frag_atoms[side][f] >> a) & 1) m |= side ? (f < GINT_SEG_COLS ? h0 : h1) : (S.fmask[0][f] & U);
        }
        const u64 mj = shfl64(m, (lane + 8) & 31);
        if (tv.diag) m = lane < 8 ? (m | mj) : 0ull;      // the atoms are evaluated once, for both sides
        if (lane < 16) S.need[lane] = m;
        if (lane == 0) { S.U = U; S.hmask[0] = h0; S.hmask[1] = h1; S.ncub = ncub; }
    } else if (warp == 1) {
        // segments: piece (row fragment r, half h) = columns [cb, cb + n); sorted by falling n and dealt to the
        // sub-partitions 0,1,2,3,3,2,1,0,... (warp w runs on sub-partition w % 4)
        if (lane < GINT_MAX_SEG) S.seg[lane] = 0;
        __syncwarp();
        int pn = 0, pcb = 0;
        const int r = lane >> 1, h = lane & 1;
        if (lane < 2 * GINT_TILE_FRAG && r < tv.nfI) {
            const int cf = tv.diag ? (S.cstart[1][S.row_atom[0][8 * r]] >> 3) : 0;
            if (h == 0) { pcb = cf; pn = min(GINT_SEG_COLS, tv.nfJ) - cf; }
            else { pcb = max(GINT_SEG_COLS, cf); pn = tv.nfJ - pcb; }
            pn = max(pn, 0);
        }
        int rank = 0;
        for (int j = 0; j < 2 * GINT_TILE_FRAG; j++) {
            const int nj = __shfl_sync(0xffffffffu, pn, j);
            rank += (nj > pn) || (nj == pn && j < lane);
        }
        if (pn > 0) {
            const int k7 = rank & 7, s = k7 < 4 ? k7 : 7 - k7, j = 2 * (rank >> 3) + (k7 >= 4);
            const int W = GINT_MMA_WARPS / 4;         // consumer warps per sub-partition
            S.seg[s + 4 * (j % W) + GINT_MMA_WARPS * (j / W)] = r | (pcb << 8) | (pn << 16);
        }
    }
    __syncthreads();
    tv.nchunk = (S.ncub + 3) >> 2;
    if (tid == 0) {
        S.tv = tv;
        for (int s = 0; s < GINT_STAGES; s++) { mbar_init(&S.full[s], GINT_EVAL_WARPS); mbar_init(&S.empty[s], GINT_MMA_WARPS); }
    }
    __syncthreads();
}

// ---------------------------------------------------------------------------------------------------
// Stage c of a tile = its cubelets 4c .. 4c+3; lane = 8 q + p: point p = (px, py, pz) bits of the q-th cubelet.
__device__ __forceinline__ bool stage_point(const TileSmem& S, const TileView& tv, int c, int lane, int& gi, int& gj, int& gk) {
    const int ci = 4 * c + (lane >> 3), p = lane & 7;
    if (ci >= S.ncub) return false;
    const int cl = S.cub[ci];
    const int ix = 2 * (cl >> 4) + (p >> 2), iy = 2 * ((cl >> 2) & 3) + ((p >> 1) & 1), iz = 2 * (cl & 3) + (p & 1);
    gi = tv.i0 + ix; gj = tv.j0 + iy; gk = tv.k0 + iz;
    return ix < tv.ex && iy < tv.ey && iz < tv.ez;
}

// Run by one warp, two stages ahead of the evaluation that consumes them (so that the global load of V is off the
// critical path): the stage's mesh points (coordinates, vlocal weight V dV) and its compacted item list.  An item
// is (atom slot, cubelet of the stage) whose orbital rows some segment reads on that cubelet: first the items on
// which the atom is really non-zero (evaluated), then those that only need zeros.
template <bool VLOCAL>
__device__ __forceinline__ void make_stage(const Geom& g, TileSmem& S, const TileView& tv, int c, const double* __restrict__ V) {
    const int lane = threadIdx.x & 31, par = c & 1;
    int gi, gj, gk;
    double4 p = make_double4(0.0, 0.0, 0.0, 0.0);
    const bool valid = stage_point(S, tv, c, lane, gi, gj, gk);
    if (valid) {
        mesh_point(g, gi, gj, gk, p.x, p.y, p.z);
        p.w = VLOCAL ? __ldg(V + ((size_t)gi * g.N[1] + gj) * g.N[2] + gk) * g.dV : 1.0;
    }
    S.pts[par][lane] = p;
    S.valid[par][lane] = valid ? 1 : 0;
    // candidates: lane -> (slot lane >> 2, cubelet lane & 3) and (slot 8 + (lane >> 2), same cubelet)
    const int ci = 4 * c + (lane & 3);
    const bool inb = ci < S.ncub;
    const int cl = inb ? S.cub[ci] : 0;
    const int s0 = lane >> 2, s1 = 8 + s0;
    const bool n0 = inb && ((S.need[s0] >> cl) & 1ull), n1 = inb && ((S.need[s1] >> cl) & 1ull);
    const bool a0 = n0 && ((S.amask[s0] >> cl) & 1ull), a1 = n1 && ((S.amask[s1] >> cl) & 1ull);
    const unsigned e0 = __ballot_sync(0xffffffffu, a0), e1 = __ballot_sync(0xffffffffu, a1);
    const unsigned z0 = __ballot_sync(0xffffffffu, n0 && !a0), z1 = __ballot_sync(0xffffffffu, n1 && !a1);
    const unsigned lt = (1u << lane) - 1u;
    const int ne = __popc(e0) + __popc(e1);
    if (a0) S.item[par][__popc(e0 & lt)] = (unsigned char)lane;
    else if (n0) S.item[par][ne + __popc(z0 & lt)] = (unsigned char)lane;
    if (a1) S.item[par][__popc(e0) + __popc(e1 & lt)] = (unsigned char)(32 + lane);
    else if (n1) S.item[par][ne + __popc(z0) + __popc(z1 & lt)] = (unsigned char)(32 + lane);
    if (lane == 0) { S.neval[par] = ne; S.nitem[par] = ne + __popc(z0) + __popc(z1); }
}

// ---------------------------------------------------------------------------------------------------
// Orbital evaluation of one stage (north_star step 2): a quarter warp = one item, lane p = point p of the cubelet.
// phi = R_s(|d|) Y_lm(d/|d|), zero for |d| >= rc (Fig. 6); radial part: per-interval
// cubic in b = r/dr - i (reading R5), coefficients read with 128-bit loads.  vlocal scales side J by V dV.
// A diagonal tile evaluates each atom once and writes both sides.
template <bool VLOCAL>
__device__ __forceinline__ void eval_stage(const Geom& g, TileSmem& S, const TileView& tv, int ps, int st, int rank,
                                           const double* __restrict__ tab) {   // ps: ring slot of phi; st: parity of the point / item lists
    const int lane = threadIdx.x & 31;
    const int nitem = S.nitem[st], neval = S.neval[st];
    const bool two = tv.diag;
    for (int base = 4 * rank; base < nitem; base += 4 * GINT_EVAL_WARPS) {
        const int idx = base + (lane >> 3);
        const bool on = idx < nitem;
        const int it = on ? S.item[st][idx] : 0;
        const int slot = it >> 2, col = 8 * (it & 3) + (lane & 7);
        const int side = slot >> 3, a = slot & 7;
        double* o0 = &S.phi[ps][side][S.cstart[side][a]][col];
        double* o1 = &S.phi[ps][1][S.cstart[side][a]][col];
        if (base >= neval) {                        // the four items only need zeros
            const int norb = on ? S.cstart[side][a + 1] - S.cstart[side][a] : 0;
            for (int o = 0; o < norb; o++) { o0[o * GINT_LD] = 0.0; if (two) o1[o * GINT_LD] = 0.0; }
            continue;
        }
        const SlotInfo si = S.sinfo[slot];
        const double4 P = S.pts[st][col];
        const double dx = P.x - S.pos[slot][0], dy = P.y - S.pos[slot][1], dz = P.z - S.pos[slot][2];
        const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
        const bool inside = on && idx < neval && S.valid[st][col] && r2 < si.rc2;
        // lanes outside the sphere run the same instructions on a clamped radius and store zeros
        const double w0 = inside ? ((VLOCAL && side) ? P.w : 1.0) : 0.0;
        const double w1 = inside ? (VLOCAL ? P.w : 1.0) : 0.0;
        // 1/r by two Newton steps from the single-precision reciprocal square root (relative error ~1e-7 -> 1e-14 -> 1e-28)
        const double q = fmin(fmax(r2, 1e-30), si.rc2);
        double ir = (double)rsqrtf((float)q);
        ir = ir * fma(-0.5 * q, ir * ir, 1.5);
        ir = ir * fma(-0.5 * q, ir * ir, 1.5);
        const double r = q * ir;
        const int nsh = on ? si.nsh : 0;
        const double x = r * g.inv_dr;
        int i = (int)x;
        i = min(i, si.n_int - 1);
        const double bq = x - (double)i;
        const double2* row = reinterpret_cast<const double2*>(tab) + ((size_t)si.tab_off + (size_t)i * si.nsh) * 2;
        const bool tiny = r < 1e-12;
        if (tiny) ir = 0.0;
        const double ux = dx * ir, uy = dy * ir, uz = dz * ir;
        const double lz = tiny ? 0.0 : 1.0;          // l > 0 orbitals vanish at the nucleus
#define GINT_PUT(v) do { const double v_ = (v); *o0 = w0 * v_; o0 += GINT_LD; if (two) { *o1 = w1 * v_; o1 += GINT_LD; } } while (0)
        for (int k0 = 0; k0 < nsh; k0 += GINT_EVAL_GROUP) {
            double2 c01[GINT_EVAL_GROUP], c23[GINT_EVAL_GROUP];
#pragma unroll
            for (int u = 0; u < GINT_EVAL_GROUP; u++)
                if (k0 + u < nsh) { c01[u] = __ldg(row + 2 * (k0 + u)); c23[u] = __ldg(row + 2 * (k0 + u) + 1); }
#pragma unroll
            for (int u = 0; u < GINT_EVAL_GROUP; u++) {
                if (k0 + u >= nsh) break;
                const double R = fma(fma(fma(c23[u].y, bq, c23[u].x), bq, c01[u].y), bq, c01[u].x);
                const int l = (si.lpack >> (2 * (k0 + u))) & 3;
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
        }
#undef GINT_PUT
    }
}

// ---------------------------------------------------------------------------------------------------
// Producer / consumer plumbing.  Warp groups 2,3 (producers) evaluate orbital values into a ring of GINT_STAGES
// shared-memory stages; warp groups 0,1 (consumers) run the DMMA chains.  full[s] completes when all producer warps
// have written stage s, empty[s] when all consumer warps have read it.  setmaxnreg moves registers from the
// producers (80 per thread) to the consumers (176), which hold the whole 104 x 104 block.
__device__ __forceinline__ void mbar_arrive(u64* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(u64* bar, int parity) {
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}"
                 :: "r"(a), "r"(parity) : "memory");
}
__device__ __forceinline__ void producer_sync() { asm volatile("bar.sync 1, %0;" :: "n"(32 * GINT_EVAL_WARPS) : "memory"); }

// Segments of a consumer warp.
struct Seg {
    int w;                           // row fragment | first column fragment << 8 | column fragments << 16 (0 = unused)
    u64 act;                         // cubelets on which the row fragment and some column fragment are both active
    __device__ __forceinline__ int row() const { return w & 255; }
    __device__ __forceinline__ int cb() const { return (w >> 8) & 255; }
    __device__ __forceinline__ int n() const { return w >> 16; }
};
__device__ __forceinline__ Seg load_seg(const TileSmem& S, int slot) {
    Seg s; s.w = S.seg[slot];
    u64 cm = 0;
    for (int j = 0; j < s.n(); j++) cm |= S.fmask[1][s.cb() + j];
    s.act = s.n() ? (S.fmask[0][s.row()] & cm) : 0ull;
    return s;
}
// 4-bit activity of a segment on the cubelets of stage c
__device__ __forceinline__ unsigned stage_bits(const TileSmem& S, int c, u64 act) {
    const unsigned cw = *reinterpret_cast<const unsigned*>(&S.cub[4 * c]);
    const int nq = min(4, S.ncub - 4 * c);
    unsigned bits = 0;
#pragma unroll
    for (int q = 0; q < 4; q++) bits |= (unsigned)((act >> ((cw >> (8 * q)) & 63u)) & 1ull) << q;
    return bits & ((1u << nq) - 1u);
}

// vlocal: acc[j] += Phi_I[row fragment]^T-slice x (V dV Phi_J)[column fragment cb + j] over the 8 points of every
// active cubelet of the stage: one 128-bit shared load per operand fragment (points 2 lc, 2 lc + 1 of the lane's
// orbital row) feeds two DMMA k-steps (k index lc <-> point 2 lc, then point 2 lc + 1).
template <int N>
__device__ __forceinline__ void vl_seg(double (&acc)[GINT_SEG_COLS][2], unsigned pa, unsigned pb, unsigned bits) {
#pragma unroll
    for (int q = 0; q < 4; q++) {
        if (!((bits >> q) & 1u)) continue;
        const double2 a = lds128(pa + 64 * q);
        double2 bv[N];
#pragma unroll
        for (int j = 0; j < N; j++) bv[j] = lds128(pb + (j * 8 * GINT_LD + 8 * q) * 8);
#pragma unroll
        for (int j = 0; j < N; j++) dmma884(acc[j], a.x, bv[j].x);
#pragma unroll
        for (int j = 0; j < N; j++) dmma884(acc[j], a.y, bv[j].y);
    }
}
__device__ __forceinline__ void vl_seg_dispatch(int n, double (&acc)[GINT_SEG_COLS][2], unsigned pa, unsigned pb, unsigned bits) {
    switch (n) {
        case 7: vl_seg<7>(acc, pa, pb, bits); break;
        case 6: vl_seg<6>(acc, pa, pb, bits); break;
        case 5: vl_seg<5>(acc, pa, pb, bits); break;
        case 4: vl_seg<4>(acc, pa, pb, bits); break;
        case 3: vl_seg<3>(acc, pa, pb, bits); break;
        case 2: vl_seg<2>(acc, pa, pb, bits); break;
        case 1: vl_seg<1>(acc, pa, pb, bits); break;
        default: break;
    }
}

// producer loop shared by both kernels: stage c of the tile goes to ring slot c % GINT_STAGES
template <bool VLOCAL>
__device__ __forceinline__ void producer_loop(const Geom& g, TileSmem& S, int nchunk, const double* __restrict__ tab, const double* __restrict__ V) {
    const int pw = (threadIdx.x >> 5) - GINT_MMA_WARPS;
    const TileView& tv = S.tv;
    if (pw == 0) make_stage<VLOCAL>(g, S, tv, 0, V);
    for (int c = 0; c < nchunk; c++) {
        const int s = c % GINT_STAGES, k = c / GINT_STAGES;
        producer_sync();              // the point / item lists of stage c are complete; all producers are done with stage c-1
        if (pw == (c + 1) % GINT_EVAL_WARPS) make_stage<VLOCAL>(g, S, tv, c + 1, V);
        if (k > 0) mbar_wait(&S.empty[s], (k - 1) & 1);
        eval_stage<VLOCAL>(g, S, tv, s, c & 1, pw, tab);
        __syncwarp();
        if ((threadIdx.x & 31) == 0) mbar_arrive(&S.full[s]);
    }
}

// ---------------------------------------------------------------------------------------------------
// gint_vlocal main kernel (north_star step 3a): W_IJ = Phi_I^T diag(V dV) Phi_J accumulated over the whole batch in
// DMMA accumulators, then added to the canonical-half value array with fp64 reductions (red.global.add.f64):
// one reduction per element per batch.
__global__ void __launch_bounds__(GINT_THREADS, 1)
k_vlocal_tile(Geom g, const int2* __restrict__ tile, const int* __restrict__ bstart, const NeighEntry* __restrict__ bent,
              const double* __restrict__ atom_pos, const int* __restrict__ atom_spec, const SpeciesDev* __restrict__ sp,
              const double* __restrict__ tab, const int* __restrict__ crow, const u64* __restrict__ ckey,
              const unsigned int* __restrict__ coff, const double* __restrict__ V, double* __restrict__ Hc) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TileSmem& S = *reinterpret_cast<TileSmem*>(smem_raw);
    {
        TileView tv0;
        tile_setup(g, S, tv0, tile, bstart, bent, atom_pos, atom_spec, sp, crow, ckey, coff);
    }
    const int nchunk = S.tv.nchunk;
    if (nchunk == 0) return;
    const int warp = threadIdx.x >> 5;
    if (warp >= GINT_MMA_WARPS) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" :: "n"(GINT_REGS_EVAL));
        producer_loop<true>(g, S, nchunk, tab, V);
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" :: "n"(GINT_REGS_MMA));
    const int lane = threadIdx.x & 31, lr = lane >> 2, lc = lane & 3;
    Seg sg[GINT_WARP_SEGS];
    double acc[GINT_WARP_SEGS][GINT_SEG_COLS][2];
#pragma unroll
    for (int k = 0; k < GINT_WARP_SEGS; k++) {
        sg[k] = load_seg(S, warp + GINT_MMA_WARPS * k);
#pragma unroll
        for (int j = 0; j < GINT_SEG_COLS; j++) { acc[k][j][0] = 0.0; acc[k][j][1] = 0.0; }
    }
    for (int c = 0; c < nchunk; c++) {
        const int s = c % GINT_STAGES;
        mbar_wait(&S.full[s], (c / GINT_STAGES) & 1);
        const unsigned pa = smem_addr(&S.phi[s][0][lr][2 * lc]), pb = smem_addr(&S.phi[s][1][lr][2 * lc]);
#pragma unroll
        for (int k = 0; k < GINT_WARP_SEGS; k++) {
            const unsigned bits = stage_bits(S, c, sg[k].act);
            if (bits) vl_seg_dispatch(sg[k].n(), acc[k], pa + sg[k].row() * (64 * GINT_LD), pb + sg[k].cb() * (64 * GINT_LD), bits);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&S.empty[s]);
    }
    // flush: element (row, col) -> atom pair (a, b), orbitals (oa, ob) -> canonical block (transposed if the canonical
    // key is (b, a)).  Exact zeros (fragments never touched, atoms that do not overlap inside this batch) are skipped.
#pragma unroll
    for (int k = 0; k < GINT_WARP_SEGS; k++) {
        if (sg[k].n() == 0 || sg[k].act == 0ull) continue;
        const int row = 8 * sg[k].row() + lr;
        const int a = S.row_atom[0][row], oa = S.row_orb[0][row];
        if (a == 255) continue;
#pragma unroll
        for (int j = 0; j < GINT_SEG_COLS; j++) {
            if (j >= sg[k].n()) break;
#pragma unroll
            for (int e = 0; e < 2; e++) {
                const double v = acc[k][j][e];
                const int col = 8 * (sg[k].cb() + j) + 2 * lc + e;
                const int bb = S.row_atom[1][col], ob = S.row_orb[1][col];
                if (bb == 255 || v == 0.0) continue;
                const PairEnt pe = S.pair[a][bb];
                if (pe.off == 0xffffffffu) continue;
                atomicAdd(Hc + pe.off + oa * pe.sr + ob * pe.sc, v);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// gint_rho main kernel (north_star step 3b).  The density blocks Dh_IJ of the tile are stationary DMMA A operands
// (registers): per cubelet X^T = Dh_seg^T Phi_I (8 orbitals of J x 8 points per column fragment) and
// rho_g += sum_j X_jg Phi_J,jg.  Dh = canonical-half, symmetrised density blocks (k_sym_D).
template <int N>
__device__ __forceinline__ void rho_cols(const double (&d)[GINT_SEG_COLS][2], int j0, double b0, double b1, unsigned pj, double& p0, double& p1) {
    double2 f[N];
#pragma unroll
    for (int j = 0; j < N; j++) f[j] = lds128(pj + ((j0 + j) * 8 * GINT_LD) * 8);
    double x[N][2];
#pragma unroll
    for (int j = 0; j < N; j++) { x[j][0] = 0.0; x[j][1] = 0.0; dmma884(x[j], d[j0 + j][0], b0); }
#pragma unroll
    for (int j = 0; j < N; j++) dmma884(x[j], d[j0 + j][1], b1);
#pragma unroll
    for (int j = 0; j < N; j++) { p0 = fma(x[j][0], f[j].x, p0); p1 = fma(x[j][1], f[j].y, p1); }
}
template <int N>
__device__ __forceinline__ void rho_seg(const double (&d)[GINT_SEG_COLS][2], unsigned pi, unsigned pj, unsigned bits, double (&part)[4][2]) {
#pragma unroll
    for (int q = 0; q < 4; q++) {
        if (!((bits >> q) & 1u)) continue;
        const double b0 = lds64(pi + 64 * q), b1 = lds64(pi + (4 * GINT_LD + 8 * q) * 8);       // Phi_I[8 row + lc (+4)][point 8q + lr]
        constexpr int N0 = N > 4 ? 4 : N;
        rho_cols<N0>(d, 0, b0, b1, pj + 64 * q, part[q][0], part[q][1]);
        if (N > 4) rho_cols<(N > 4 ? N - 4 : 1)>(d, 4, b0, b1, pj + 64 * q, part[q][0], part[q][1]);
    }
}
__device__ __forceinline__ void rho_seg_dispatch(int n, const double (&d)[GINT_SEG_COLS][2], unsigned pi, unsigned pj,
                                                 unsigned bits, double (&part)[4][2]) {
    switch (n) {
        case 7: rho_seg<7>(d, pi, pj, bits, part); break;
        case 6: rho_seg<6>(d, pi, pj, bits, part); break;
        case 5: rho_seg<5>(d, pi, pj, bits, part); break;
        case 4: rho_seg<4>(d, pi, pj, bits, part); break;
        case 3: rho_seg<3>(d, pi, pj, bits, part); break;
        case 2: rho_seg<2>(d, pi, pj, bits, part); break;
        case 1: rho_seg<1>(d, pi, pj, bits, part); break;
        default: break;
    }
}
// stationary operand of a segment: d[j][h] = Dh[orbital row 8 row + 4h + lc of I][orbital column 8 (cb + j) + lr of J]
__device__ __forceinline__ void load_dseg(const TileSmem& S, const Seg& sg, const double* __restrict__ Dh, double (&d)[GINT_SEG_COLS][2]) {
    const int lane = threadIdx.x & 31, lr = lane >> 2, lc = lane & 3;
#pragma unroll
    for (int j = 0; j < GINT_SEG_COLS; j++)
#pragma unroll
        for (int h = 0; h < 2; h++) {
            double v = 0.0;
            if (j < sg.n()) {
                const int row = 8 * sg.row() + 4 * h + lc, col = 8 * (sg.cb() + j) + lr;
                const int a = S.row_atom[0][row], bb = S.row_atom[1][col];
                if (a != 255 && bb != 255) {
                    const PairEnt pe = S.pair[a][bb];
                    if (pe.off != 0xffffffffu) v = __ldg(Dh + pe.off + S.row_orb[0][row] * pe.sr + S.row_orb[1][col] * pe.sc);
                }
            }
            d[j][h] = v;
        }
}

__global__ void __launch_bounds__(GINT_THREADS, 1)
k_rho_tile(Geom g, const int2* __restrict__ tile, const int* __restrict__ bstart, const NeighEntry* __restrict__ bent,
           const double* __restrict__ atom_pos, const int* __restrict__ atom_spec, const SpeciesDev* __restrict__ sp,
           const double* __restrict__ tab, const int* __restrict__ crow, const u64* __restrict__ ckey,
           const unsigned int* __restrict__ coff, const double* __restrict__ Dh, double* __restrict__ rho) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TileSmem& S = *reinterpret_cast<TileSmem*>(smem_raw);
    {
        TileView tv0;
        tile_setup(g, S, tv0, tile, bstart, bent, atom_pos, atom_spec, sp, crow, ckey, coff);
    }
    const int nchunk = S.tv.nchunk;
    if (nchunk == 0) return;
    const int warp = threadIdx.x >> 5;
    if (warp >= GINT_MMA_WARPS) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" :: "n"(GINT_REGS_EVAL));
        producer_loop<false>(g, S, nchunk, tab, nullptr);
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" :: "n"(GINT_REGS_MMA));
    const int lane = threadIdx.x & 31, lr = lane >> 2, lc = lane & 3;
    Seg sg[GINT_WARP_SEGS];
    double d[GINT_WARP_SEGS][GINT_SEG_COLS][2];
#pragma unroll
    for (int k = 0; k < GINT_WARP_SEGS; k++) {
        sg[k] = load_seg(S, warp + GINT_MMA_WARPS * k);
        load_dseg(S, sg[k], Dh, d[k]);
    }
    for (int c = 0; c < nchunk; c++) {
        const int s = c % GINT_STAGES;
        double part[4][2];
#pragma unroll
        for (int q = 0; q < 4; q++) { part[q][0] = 0.0; part[q][1] = 0.0; }
        mbar_wait(&S.full[s], (c / GINT_STAGES) & 1);
        const unsigned pi = smem_addr(&S.phi[s][0][lc][lr]), pj = smem_addr(&S.phi[s][1][lr][2 * lc]);
        unsigned any = 0;
#pragma unroll
        for (int k = 0; k < GINT_WARP_SEGS; k++) {
            const unsigned bits = stage_bits(S, c, sg[k].act);
            any |= bits;
            if (bits) rho_seg_dispatch(sg[k].n(), d[k], pi + sg[k].row() * (64 * GINT_LD), pj + sg[k].cb() * (64 * GINT_LD), bits, part);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&S.empty[s]);
        if (!any) continue;
        // part[q][e]: points 8q + 2lc + e, partial over the lane's orbital row lr -> reduce-scatter over lr (lane bits 2..4)
        double r4[4], r2[2], r1;
        {
            const bool hi = lane & 16;
#pragma unroll
            for (int i = 0; i < 4; i++) {     // value index t = 2q + e; lanes with bit 4 clear keep t < 4
                const double keep = hi ? part[2 + (i >> 1)][i & 1] : part[i >> 1][i & 1];
                const double send = hi ? part[i >> 1][i & 1] : part[2 + (i >> 1)][i & 1];
                r4[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
            }
            const bool mid = lane & 8;
#pragma unroll
            for (int i = 0; i < 2; i++) {
                const double keep = mid ? r4[2 + i] : r4[i], send = mid ? r4[i] : r4[2 + i];
                r2[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
            }
            const bool low = lane & 4;
            const double keep = low ? r2[1] : r2[0], send = low ? r2[0] : r2[1];
            r1 = keep + __shfl_xor_sync(0xffffffffu, send, 4);
        }
        // the lane now owns point 8 (lr >> 1) + 2 lc + (lr & 1) of the stage
        int gi, gj, gk;
        if (r1 != 0.0 && stage_point(S, S.tv, c, 8 * (lr >> 1) + 2 * lc + (lr & 1), gi, gj, gk))
            atomicAdd(rho + ((size_t)gi * g.N[1] + gj) * g.N[2] + gk, r1);
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
                if (fma(dx, dx, fma(dy, dy, dz * dz)) < Sp->rc * Sp->rc) { na++; no += Sp->norb; }
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
