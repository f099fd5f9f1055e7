// gint_kernels.cu -- the per-call hot path (north_star steps 2 and 3), fp64, sm_100a.
//
// Work decomposition.  The mesh is cut into grid batches (default 8x8x16 points) whose neighbouring
// atom images were listed by gint_init, most active first, each with a 128-bit ACTIVITY MASK over the
// batch's 4x4x8 "cubelets" of 2x2x2 mesh points (bit set = some point of the cubelet lies inside the atom's cutoff
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
// activity mask over the (at most 128) cubelets of a batch
struct cmask { u64 lo, hi; };
__device__ __forceinline__ cmask operator|(cmask a, cmask b) { return cmask{a.lo | b.lo, a.hi | b.hi}; }
__device__ __forceinline__ cmask operator&(cmask a, cmask b) { return cmask{a.lo & b.lo, a.hi & b.hi}; }
__device__ __forceinline__ cmask& operator|=(cmask& a, cmask b) { a.lo |= b.lo; a.hi |= b.hi; return a; }
__device__ __forceinline__ bool cbit(const cmask& m, int i) { return ((i < 64 ? m.lo >> i : m.hi >> (i - 64)) & 1ull) != 0; }
__device__ __forceinline__ cmask czero() { return cmask{0ull, 0ull}; }
#ifndef GINT_DBG_STATS
#define DBG_T(x)
#define DBG_ADD(i, v)
#else
__device__ unsigned long long g_dbg[16];
#define DBG_T(x) const long long x = clock64()
#define DBG_ADD(i, v) do { if ((threadIdx.x & 31) == 0) atomicAdd(&g_dbg[i], (unsigned long long)(v)); } while (0)
extern "C" int gint_debug_counters(unsigned long long* out) { return (int)cudaMemcpyFromSymbol(out, g_dbg, sizeof(g_dbg)); }
#endif
#ifndef GINT_EVAL_GROUP
#define GINT_EVAL_GROUP 5          // radial shells whose spline cells are loaded together (registers vs memory-level parallelism)
#define GINT_EVAL_GROUP_RHO 2      // gint_rho's producers run with 72 registers: measured 91.9 ms (5), 88.6 (3), 87.9 (2) at cfg3
#endif

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
    double4 pts[GINT_NCUB * GINT_CPTS];                   // [cubelet id * 8 + p]: x, y, z of the batch's mesh points, weight V dV (vlocal) or 1 (rho);
                                        // points outside the mesh: far away, weight 0
    u64 full[GINT_STAGES], empty[GINT_STAGES];   // mbarriers: stage written by all producer warps / read by all consumer warps
    double pos[16][4];                  // slot s < 8: atom s of group I; slot 8 + s: atom s of group J
    SlotInfo sinfo[16];
    cmask amask[16];                      // cubelets on which the slot's atom is non-zero
    cmask need[16];                       // cubelets on which the slot's orbital rows are read by some segment
    cmask fmask[2][16];                   // [side][fragment]: OR of amask over the atoms with orbitals in the fragment
    cmask hmask[2];                       // side J: OR of fmask over the column fragments 0..6 / 7..12
    cmask U;                            // cubelets the tile walks over: (any I fragment) & (any J fragment)
    PairEnt pair[GINT_TILE_ATOMS][GINT_TILE_ATOMS];   // canonical block of (I atom a, J atom b)
    int atom[16], shift[16], spec[16];
    int cstart[2][GINT_TILE_ATOMS + 1]; // first orbital row of each atom inside its group
    u64 segWhi[GINT_MAX_SEG];           // second half (list positions 64..127) of the segments' activity words
    int seg[GINT_MAX_SEG];              // slot (consumer warp) + 8 k: row fragment | first column fragment << 8 | n columns << 16
    int ncub;
    TileView tv;                        // written by tile_setup; read from here afterwards to keep registers free
    unsigned char item[GINT_MAX_CHUNKS][16 * GINT_CUBS];         // [stage][k]: slot << 2 | cubelet of the stage
    unsigned char nitem[GINT_MAX_CHUNKS], neval[GINT_MAX_CHUNKS]; // [stage]: items of the stage, of which the first neval need a real evaluation
    unsigned char cub[GINT_NCUB + 4];          // the tile's cubelets (bit numbers of U, ascending)
    unsigned char row_atom[2][GINT_TILE_ORB];   // orbital row -> atom slot inside the group (255 = padding)
    unsigned char row_orb[2][GINT_TILE_ORB];    // orbital row -> orbital index inside the atom
    unsigned char frag_atoms[2][16];            // fragment -> bit mask of the atoms it holds orbitals of
};
// the radial table follows the struct in dynamic shared memory when it fits
#define GINT_SMEM_TAB_OFF ((sizeof(TileSmem) + 15) & ~(size_t)15)
size_t gint_smem_needed(gint_ctx* c, size_t limit) {
    c->tab_in_smem = GINT_SMEM_TAB_OFF + c->tab_bytes <= limit;
    return GINT_SMEM_TAB_OFF + (c->tab_in_smem ? c->tab_bytes : 0);
}

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
__device__ __forceinline__ cmask warp_orc(cmask v) { return cmask{warp_or64(v.lo), warp_or64(v.hi)}; }
__device__ __forceinline__ u64 shfl64(u64 v, int src) {
    const unsigned lo = __shfl_sync(0xffffffffu, (unsigned)v, src), hi = __shfl_sync(0xffffffffu, (unsigned)(v >> 32), src);
    return (u64)lo | ((u64)hi << 32);
}

// ---------------------------------------------------------------------------------------------------
// Stage c of a tile = its cubelets 4c .. 4c+3; point index 8 q + p: point p = (px, py, pz) bits of the q-th cubelet.
__device__ __forceinline__ bool stage_point(const TileSmem& S, int c, int pt, int& gi, int& gj, int& gk) {
    const int ci = GINT_CUBS * c + pt / GINT_CPTS, p = pt % GINT_CPTS;
    if (ci >= S.ncub) return false;
    const int cl = S.cub[ci];
    const int ix = 2 * (cl / (4 * GINT_NCZ)) + p / (2 * GINT_CZ), iy = 2 * ((cl / GINT_NCZ) & 3) + ((p / GINT_CZ) & 1), iz = GINT_CZ * (cl % GINT_NCZ) + p % GINT_CZ;
    gi = S.tv.i0 + ix; gj = S.tv.j0 + iy; gk = S.tv.k0 + iz;
    return ix < S.tv.ex && iy < S.tv.ey && iz < S.tv.ez;
}

// Item list of stage c (tile set-up, one warp per stage).  An item is (atom slot, cubelet of the stage) whose orbital
// rows some segment reads on that cubelet: first the items on which the atom is really non-zero (evaluated), then
// those that only need zeros.
__device__ __forceinline__ void make_items(TileSmem& S, int c) {
    const int lane = threadIdx.x & 31;
    // candidates (slot, cubelet of the stage): 16 * GINT_CUBS of them, NR per lane
    constexpr int NR = (16 * GINT_CUBS + 31) / 32;
    bool act[NR], need[NR];
    unsigned eb[NR], zb[NR];
    int ne = 0, nz = 0;
#pragma unroll
    for (int r = 0; r < NR; r++) {
        const int cand = lane + 32 * r, slot = cand / GINT_CUBS, q = cand % GINT_CUBS;
        const int ci = GINT_CUBS * c + q;
        const bool inb = cand < 16 * GINT_CUBS && ci < S.ncub;
        const int cl = inb ? S.cub[ci] : 0;
        need[r] = inb && cbit(S.need[slot & 15], cl);
        act[r] = need[r] && cbit(S.amask[slot & 15], cl);
        eb[r] = __ballot_sync(0xffffffffu, act[r]);
        zb[r] = __ballot_sync(0xffffffffu, need[r] && !act[r]);
        ne += __popc(eb[r]); nz += __popc(zb[r]);
    }
    const unsigned lt = (1u << lane) - 1u;
    int pe = 0, pz = ne;
#pragma unroll
    for (int r = 0; r < NR; r++) {
        const int cand = lane + 32 * r;
        const unsigned char code = (unsigned char)(((cand / GINT_CUBS) << 2) | (cand % GINT_CUBS));
        if (act[r]) S.item[c][pe + __popc(eb[r] & lt)] = code;
        else if (need[r]) S.item[c][pz + __popc(zb[r] & lt)] = code;
        pe += __popc(eb[r]); pz += __popc(zb[r]);
    }
    if (lane == 0) { S.neval[c] = (unsigned char)ne; S.nitem[c] = (unsigned char)(ne + nz); }
}

// ---------------------------------------------------------------------------------------------------
// Orbital evaluation of one stage by one producer warp (north_star step 2): a quarter warp = one item, lane p = point
// p of the cubelet.  phi = R_s(|d|) Y_lm(d/|d|), zero for |d| >= rc (Fig. 6); radial part
// (reading R5): R = a y_i + b y_{i+1} + (a^3-a) z_i + (b^3-b) z_{i+1} from the knot cells {y, z} of the interval,
// read with 128-bit loads (from the shared-memory copy of the table when it fits).  vlocal scales side J by V dV.
// A diagonal tile evaluates each atom once and writes both sides.  `first`: this warp's first item of the stage.
template <bool VLOCAL>
__device__ __forceinline__ void eval_stage(const Geom& g, TileSmem& S, int ps, int c, int first, const double2* __restrict__ tab,
                                           const double* __restrict__ V) {
    const int lane = threadIdx.x & 31;
    constexpr int GROUP = VLOCAL ? GINT_EVAL_GROUP : GINT_EVAL_GROUP_RHO;
    const int nitem = S.nitem[c], neval = S.neval[c];
    const bool two = VLOCAL && S.tv.diag;      // gint_rho reads side I twice in a diagonal tile instead
    for (int base = first; base < nitem; base += (32 / GINT_CPTS) * GINT_EVAL_WARPS) {
        const int idx = base + lane / GINT_CPTS;
        const bool on = idx < nitem;
        const int it = on ? S.item[c][idx] : 0;
        const int slot = it >> 2, pt = GINT_CPTS * (it & 3) + lane % GINT_CPTS;
        const int side = slot >> 3, a = slot & 7;
        double* o0 = &S.phi[ps][side][S.cstart[side][a]][pt];
        if (base >= neval) {                        // the four items only need zeros
            const int norb = on ? S.cstart[side][a + 1] - S.cstart[side][a] : 0;
            for (int o = 0; o < norb; o++) { o0[o * GINT_LD] = 0.0; if (two) o0[o * GINT_LD + GINT_TILE_ORB * GINT_LD] = 0.0; }
            continue;
        }
        const double4 P = S.pts[GINT_CPTS * S.cub[min(GINT_CUBS * c + (it & 3), GINT_NCUB - 1)] + lane % GINT_CPTS];
        const double wv = P.w;
        const SlotInfo si = S.sinfo[slot];
        const double dx = P.x - S.pos[slot][0], dy = P.y - S.pos[slot][1], dz = P.z - S.pos[slot][2];
        const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
        const bool inside = on && idx < neval && r2 < si.rc2;
        // 1/r by one Newton step from the single-precision reciprocal square root: relative error 2.4e-7 -> 1.5 e^2 = 9e-14,
        // three orders below the 1e-10 parity bar (a second step would cost four more dependent FP64 operations)
        const double q = fmin(fmax(r2, 1e-30), si.rc2);
        double ir = (double)rsqrtf((float)q);
        ir = ir * fma(-0.5 * q, ir * ir, 1.5);
        const double r = q * ir;
        const int nsh = on ? si.nsh : 0;
        const double x = r * g.inv_dr;
        int i = (int)x;
        i = min(i, si.n_int - 1);
        const double b = x - (double)i, am = 1.0 - b;
        const double a3 = (am * am - 1.0) * am, b3 = (b * b - 1.0) * b;
        const double2* row = tab + (si.tab_off + i * si.nsh);
        const bool tiny = r < 1e-12;
        if (tiny) ir = 0.0;
        // lanes outside the sphere run the same instructions on a clamped radius and store zeros
        const double w0 = inside ? ((VLOCAL && side) ? wv : 1.0) : 0.0;
        const double w1 = inside ? wv : 0.0;
        const double ux = dx * ir, uy = dy * ir, uz = dz * ir;
        // Angular factors times the store weight, all independent of the radial values: the FP64 pipe is shared with the
        // consumers' DMMAs, under which a DEPENDENT FP64 operation costs ~25 cycles but independent ones overlap (measured),
        // so the evaluation is written as wide as the registers allow: every output is then one multiply R_k * yw[m].
        double yw[9];
        {
            const double c1 = 0.4886025119029199 * w0, c2 = (tiny ? 0.0 : 1.0925484305920792) * w0;     // l > 0 orbitals vanish at the nucleus
            const double c20 = (tiny ? 0.0 : 0.31539156525252005) * w0, c22 = (tiny ? 0.0 : 0.5462742152960396) * w0;
            const double c2x = c2 * ux, c2y = c2 * uy;
            yw[0] = 0.28209479177387814 * w0;
            yw[1] = c1 * uy; yw[2] = c1 * uz; yw[3] = c1 * ux;
            yw[4] = c2x * uy; yw[5] = c2y * uz; yw[6] = c20 * fma(3.0 * uz, uz, -1.0); yw[7] = c2x * uz; yw[8] = c22 * fma(ux, ux, -uy * uy);
        }
        const double wr = (two && inside) ? (VLOCAL ? wv : 1.0) : 0.0;      // diagonal tile: side J = wr / w0-scaled copy (w0 = 1 inside)
#define GINT_PUT(m) do { const double v_ = R * yw[m]; *o0 = v_; if (two) o0[GINT_TILE_ORB * GINT_LD] = wr * v_; o0 += GINT_LD; } while (0)
        for (int k0 = 0; k0 < nsh; k0 += GROUP) {
            double Rk[GROUP];
#pragma unroll
            for (int u = 0; u < GROUP; u++) {
                Rk[u] = 0.0;
                if (k0 + u < nsh) {
                    const double2 c0 = row[k0 + u], c1 = row[nsh + k0 + u];
                    Rk[u] = fma(am, c0.x, fma(b, c1.x, fma(a3, c0.y, b3 * c1.y)));
                }
            }
#pragma unroll
            for (int u = 0; u < GROUP; u++) {
                if (k0 + u >= nsh) break;
                const double R = Rk[u];
                const int l = (si.lpack >> (2 * (k0 + u))) & 3;
                if (l == 0) {
                    GINT_PUT(0);
                } else if (l == 1) {
                    GINT_PUT(1); GINT_PUT(2); GINT_PUT(3);
                } else {
                    GINT_PUT(4); GINT_PUT(5); GINT_PUT(6); GINT_PUT(7); GINT_PUT(8);
                }
            }
        }
#undef GINT_PUT
    }
}

// ---------------------------------------------------------------------------------------------------
// Tile set-up: atom slots, orbital-row maps, canonical block of every atom pair of the tile, activity masks,
// cubelet list, segments.
__device__ __forceinline__ void tile_setup(const Geom& g, TileSmem& S, TileView& tv, const int2* __restrict__ tile,
                                           const int* __restrict__ bstart, const NeighEntry* __restrict__ bent,
                                           const double* __restrict__ atom_pos, const int* __restrict__ atom_spec,
                                           const SpeciesDev* __restrict__ sp, const int* __restrict__ crow,
                                           const u64* __restrict__ ckey, const unsigned int* __restrict__ coff,
                                           const double* __restrict__ tab, int tab_cells, const double* __restrict__ V) {
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    DBG_T(ts0);
    const int2 td = tile[blockIdx.x];            // head of the dependent chain tile -> batch -> neighbour entries -> atoms: issue it first
    // copy of the radial table (tab_cells = 0: it stays in global memory): 8 independent 16-byte loads per thread in flight
    {
        const double2* src = reinterpret_cast<const double2*>(tab);
        double2* dst = reinterpret_cast<double2*>(reinterpret_cast<unsigned char*>(&S) + GINT_SMEM_TAB_OFF);
        for (int i0 = tid; i0 < tab_cells; i0 += 8 * GINT_THREADS) {
            double2 tmp[8];
#pragma unroll
            for (int u = 0; u < 8; u++) if (i0 + u * GINT_THREADS < tab_cells) tmp[u] = __ldg(src + i0 + u * GINT_THREADS);
#pragma unroll
            for (int u = 0; u < 8; u++) if (i0 + u * GINT_THREADS < tab_cells) dst[i0 + u * GINT_THREADS] = tmp[u];
        }
    }
    if (tid == GINT_THREADS - 32) for (int s = 0; s < GINT_STAGES; s++) { mbar_init(&S.full[s], GINT_EVAL_WARPS); mbar_init(&S.empty[s], GINT_MMA_WARPS); }
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

    for (int q = tid; q < GINT_NCUB * GINT_CPTS; q += GINT_THREADS) {   // mesh points of the batch (V == nullptr: rho, weight 1)
        const int cl = q / GINT_CPTS, pp = q % GINT_CPTS;
        const int ix = 2 * (cl / (4 * GINT_NCZ)) + pp / (2 * GINT_CZ), iy = 2 * ((cl / GINT_NCZ) & 3) + ((pp / GINT_CZ) & 1), iz = GINT_CZ * (cl % GINT_NCZ) + pp % GINT_CZ;
        double4 P = make_double4(1e30, 0.0, 0.0, 0.0);
        if (ix < tv.ex && iy < tv.ey && iz < tv.ez) {
            const int gi = tv.i0 + ix, gj = tv.j0 + iy, gk = tv.k0 + iz;
            mesh_point(g, gi, gj, gk, P.x, P.y, P.z);
            P.w = V ? __ldg(V + ((size_t)gi * g.N[1] + gj) * g.N[2] + gk) * g.dV : 1.0;
        }
        S.pts[q] = P;
    }
    if (tid < 16) {
        const int side = tid >> 3, a = tid & 7;
        const bool valid = a < (side ? tv.nJ : tv.nI);
        int atom = 0, shift = pack_shift(0, 0, 0), spec = 0;
        double x = 0, y = 0, z = 0;
        cmask m = czero();
        if (valid) {
            const NeighEntry e = bent[e0 + (side ? eJ : eI) + a];
            int t1, t2, t3; unpack_shift(e.shift, t1, t2, t3);
            atom = e.atom; shift = e.shift; spec = atom_spec[atom]; m = cmask{e.mask[0], e.mask[1]};
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
        // first orbital row of each atom inside its group: prefix sum of norb over the 8 lanes of the side
        const int norb = valid ? Sp->norb : 0;
        int inc = norb;
#pragma unroll
        for (int dlt = 1; dlt < 8; dlt <<= 1) { const int t = __shfl_up_sync(0xffffu, inc, dlt, 8); if (a >= dlt) inc += t; }
        S.cstart[side][a] = inc - norb;
        if (a == 7) S.cstart[side][8] = inc;
    }
    DBG_T(ts1);
    __syncthreads();
    DBG_T(ts2);
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
        cmask fm = czero();
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
    DBG_T(ts3);
    if (warp == 0 || warp == 2) {
        // union masks (both warps), then warp 0: cubelet list; warp 2: per-slot read sets
        const cmask vI = lane < tv.nfI ? S.fmask[0][lane] : czero();
        const cmask vJ = lane < tv.nfJ ? S.fmask[1][lane] : czero();
        const cmask anyI = warp_orc(vI);
        const cmask h0 = warp_orc(lane < GINT_SEG_COLS ? vJ : czero()) & anyI, h1 = warp_orc(lane >= GINT_SEG_COLS ? vJ : czero()) & anyI;
        const cmask U = h0 | h1;
        if (warp == 0) {
            const unsigned Uw[4] = {(unsigned)U.lo, (unsigned)(U.lo >> 32), (unsigned)U.hi, (unsigned)(U.hi >> 32)};
            const unsigned lt = (1u << lane) - 1u;
            int before = 0;
#pragma unroll
            for (int wd = 0; wd < 4; wd++) {
                if ((Uw[wd] >> lane) & 1u) S.cub[before + __popc(Uw[wd] & lt)] = (unsigned char)(32 * wd + lane);
                before += __popc(Uw[wd]);
            }
            const int ncub = before;
            if (lane < 4) S.cub[ncub + lane] = 0;
            if (lane == 0) { S.U = U; S.hmask[0] = h0; S.hmask[1] = h1; S.ncub = ncub; }
        } else {
            cmask m = czero();
            if (lane < 16) {
                const int side = lane >> 3, a = lane & 7;
                const int nf = side ? tv.nfJ : tv.nfI;
                for (int f = 0; f < nf; f++)
                    if ((S.frag_atoms[side][f] >> a) & 1) m |= side ? (f < GINT_SEG_COLS ? h0 : h1) : (S.fmask[0][f] & U);
            }
            const cmask mj = cmask{shfl64(m.lo, (lane + 8) & 31), shfl64(m.hi, (lane + 8) & 31)};
            if (tv.diag) m = lane < 8 ? (m | mj) : czero();      // the atoms are evaluated once, for both sides
            if (lane < 16) S.need[lane] = m;
        }
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
    DBG_T(ts4);
    tv.nchunk = (S.ncub + GINT_CUBS - 1) / GINT_CUBS;
    for (int c = warp; c < tv.nchunk; c += GINT_WARPS) make_items(S, c);
    if (tid == GINT_THREADS - 1) S.tv = tv;      // a thread of the last warp: it has no item list to make (<= 16 stages, warp 15 only for 64 cubelets)
    __syncthreads();
    DBG_T(ts5); DBG_ADD(12, ts1 - ts0); DBG_ADD(13, ts2 - ts1); DBG_ADD(14, ts3 - ts2); DBG_ADD(15, ts4 - ts3); DBG_ADD(0, ts5 - ts4);
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

// Segments of a consumer warp.
#define GINT_ROWB (GINT_LD * 8)                    // bytes of one orbital row of a stage
#define GINT_SIDEB (GINT_TILE_ORB * GINT_ROWB)     // bytes of one side of a stage
#define GINT_STAGEB (2 * GINT_SIDEB)
struct Seg {
    unsigned oa;                     // byte offset of the row fragment in side I (row 8 row) | column fragments << 24 (0 = unused)
    unsigned ob;                     // byte offset of the first column fragment in side J, relative to the stage
    u64 W;                           // activity on the tile's cubelet list: bit p = the segment works on cubelet cub[p]
    int w;                           // row fragment | first column fragment << 8 | column fragments << 16
    __device__ __forceinline__ int row() const { return w & 255; }
    __device__ __forceinline__ int cb() const { return (w >> 8) & 255; }
    __device__ __forceinline__ int n() const { return w >> 16; }
};
__device__ __forceinline__ Seg load_seg(TileSmem& S, int slot, bool j_is_i = false) {   // j_is_i: column operands from side I (rho, diagonal tile)
    const int lane = threadIdx.x & 31;
    Seg s; s.w = S.seg[slot];
    cmask cm = czero();
    for (int j = 0; j < s.n(); j++) cm |= S.fmask[1][s.cb() + j];
    const cmask act = s.n() ? (S.fmask[0][s.row()] & cm) : czero();     // cubelets on which the row fragment and some column fragment are active
    unsigned wb[4];
#pragma unroll
    for (int wd = 0; wd < 4; wd++) {
        const int pp = 32 * wd + lane;
        wb[wd] = __ballot_sync(0xffffffffu, pp < S.ncub && cbit(act, S.cub[min(pp, GINT_NCUB - 1)]));
    }
    s.W = (u64)wb[0] | ((u64)wb[1] << 32);
    if (lane == 0) S.segWhi[slot] = (u64)wb[2] | ((u64)wb[3] << 32);      // list positions 64..127: fetched when the tile gets there
    __syncwarp();
    s.oa = (unsigned)(s.row() * 8 * GINT_ROWB);
    s.ob = (unsigned)((j_is_i ? 0 : GINT_SIDEB) + s.cb() * 8 * GINT_ROWB);
    return s;
}

// activity of a segment on the 8-point DMMA steps of stage c (a 16-point cubelet is two steps)
__device__ __forceinline__ unsigned stage_steps(u64 W, int c) {
    const unsigned b = (unsigned)(W >> ((GINT_CUBS * c) & 63)) & ((1u << GINT_CUBS) - 1u);
    return GINT_CPTS == 8 ? b : ((b & 1u) * 3u) | ((b & 2u) * 6u);
}
__device__ __forceinline__ void next_cubelet(unsigned& rem, unsigned pa, unsigned pb, unsigned& oa, unsigned& ob) {
    asm volatile("{\n\t.reg .u32 t, u;\n\tbrev.b32 t, %0;\n\tclz.b32 t, t;\n\tshl.b32 t, t, 6;\n\tadd.u32 %1, %3, t;\n\tadd.u32 %2, %4, t;\n\t"
                 "add.u32 u, %0, -1;\n\tand.b32 %0, %0, u;\n\t}" : "+r"(rem), "=r"(oa), "=r"(ob) : "r"(pa), "r"(pb));
}
template <int N>
__device__ __forceinline__ void vl_seg(double (&acc)[GINT_SEG_COLS][2], unsigned pa, unsigned pb, unsigned bits) {
    double ax, ay, bx[N], by[N];
    unsigned rem = bits, oa, ob;
    next_cubelet(rem, pa, pb, oa, ob);
    ax = lds64(oa);
#pragma unroll
    for (int j = 0; j < N; j++) bx[j] = lds64(ob + j * 8 * GINT_ROWB);
    ay = lds64(oa + 32);
#pragma unroll
    for (int j = 0; j < N; j++) by[j] = lds64(ob + j * 8 * GINT_ROWB + 32);
    bool more = rem != 0;
    next_cubelet(rem, pa, pb, oa, ob);
    while (more) {
        // the reload of an operand register follows the DMMA that read it: the loads issue in the shadow of the
        // 16-cycle DMMAs instead of in a gap between the two groups
#pragma unroll
        for (int j = 0; j < N; j++) {
            dmma884(acc[j], ax, bx[j]);
            bx[j] = lds64(ob + j * 8 * GINT_ROWB);
        }
        ax = lds64(oa);
        unsigned oa2, ob2;
#pragma unroll
        for (int j = 0; j < N; j++) {
            dmma884(acc[j], ay, by[j]);
            by[j] = lds64(ob + j * 8 * GINT_ROWB + 32);
            if (j == 0) { more = rem != 0; next_cubelet(rem, pa, pb, oa2, ob2); }
        }
        ay = lds64(oa + 32);
        oa = oa2; ob = ob2;
    }
#pragma unroll
    for (int j = 0; j < N; j++) dmma884(acc[j], ax, bx[j]);
#pragma unroll
    for (int j = 0; j < N; j++) dmma884(acc[j], ay, by[j]);
}
__device__ __forceinline__ void vl_seg_dispatch(int n, double (&acc)[GINT_SEG_COLS][2], unsigned pa, unsigned pb, unsigned bits) {
    // 7 and 6 are the lengths of all segments of a full off-diagonal tile: two compares instead of an indexed branch
    if (n == 7) { vl_seg<7>(acc, pa, pb, bits); return; }
    if (n == 6) { vl_seg<6>(acc, pa, pb, bits); return; }
    switch (n) {
        case 5: vl_seg<5>(acc, pa, pb, bits); break;
        case 4: vl_seg<4>(acc, pa, pb, bits); break;
        case 3: vl_seg<3>(acc, pa, pb, bits); break;
        case 2: vl_seg<2>(acc, pa, pb, bits); break;
        case 1: vl_seg<1>(acc, pa, pb, bits); break;
        default: break;
    }
}

// producer loop shared by both kernels: stage c of the tile goes to ring slot c % GINT_STAGES.  The producer warps do
// not synchronise with one another: each takes every 8th group of four items, rotating with the stage so that
// the remainders even out, and arrives on full[s] when its share of the stage is written.
template <bool VLOCAL>
__device__ __forceinline__ void producer_loop(const Geom& g, TileSmem& S, int nchunk, const double* __restrict__ tab, int tab_cells,
                                              const double* __restrict__ V) {
    const int pw = (threadIdx.x >> 5) - GINT_MMA_WARPS;
    const double2* tb = tab_cells ? reinterpret_cast<const double2*>(reinterpret_cast<const unsigned char*>(&S) + GINT_SMEM_TAB_OFF)
                                  : reinterpret_cast<const double2*>(tab);
    for (int c = 0; c < nchunk; c++) {
        const int s = c % GINT_STAGES, k = c / GINT_STAGES;
        DBG_T(t_p0);
        if (k > 0) mbar_wait(&S.empty[s], (k - 1) & 1);
        DBG_T(t_p1);
        DBG_ADD(10, t_p1 - t_p0);
#ifndef GINT_DBG_NO_EVAL
        eval_stage<VLOCAL>(g, S, s, c, (32 / GINT_CPTS) * ((pw + c) % GINT_EVAL_WARPS), tb, V);
#endif
        __syncwarp();
        if ((threadIdx.x & 31) == 0) mbar_arrive(&S.full[s]);
        DBG_T(t_p2);
        DBG_ADD(11, t_p2 - t_p1);
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
              const unsigned int* __restrict__ coff, int tab_cells, const double* __restrict__ V, double* __restrict__ Hc) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TileSmem& S = *reinterpret_cast<TileSmem*>(smem_raw);
    DBG_T(t_start);
    {
        TileView tv0;
        tile_setup(g, S, tv0, tile, bstart, bent, atom_pos, atom_spec, sp, crow, ckey, coff, tab, tab_cells, V);
    }
    DBG_T(t_setup);
    DBG_ADD(5, t_setup - t_start);
    const int nchunk = S.tv.nchunk;
    if (nchunk == 0) return;
    const int warp = threadIdx.x >> 5;
    if (warp >= GINT_MMA_WARPS) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" :: "n"(GINT_REGS_EVAL));
        producer_loop<true>(g, S, nchunk, tab, tab_cells, V);
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
#ifdef GINT_DBG_STATS
    {   // developer statistics: DMMA balance over the four sub-partitions (whole tile, and stage by stage)
        __shared__ int dbg_load[GINT_MAX_CHUNKS + 1][GINT_MMA_WARPS];
        int tot = 0;
        for (int c = 0; c < nchunk; c++) {
            int l = 0;
            for (int k = 0; k < GINT_WARP_SEGS; k++) l += 2 * sg[k].n() * __popc(stage_steps(sg[k].W, c));
            if (lane == 0) dbg_load[c][warp] = l;
            tot += l;
        }
        if (lane == 0) dbg_load[GINT_MAX_CHUNKS][warp] = tot;
        {   // DMMAs needed at (row fragment, column fragment, cubelet) granularity, and with trailing-column cut per cubelet
            unsigned long long fine = 0, lead = 0;
            for (int k = 0; k < GINT_WARP_SEGS; k++) {
                const cmask rm = S.fmask[0][sg[k].row()] & S.U;
                cmask seen = czero();
                for (int j = sg[k].n() - 1; j >= 0; j--) {
                    const cmask cm = S.fmask[1][sg[k].cb() + j] & rm;
                    fine += 2 * (__popcll(cm.lo) + __popcll(cm.hi));
                    seen |= cm;
                    lead += 2 * (__popcll(seen.lo) + __popcll(seen.hi));      // columns 0..j computed wherever some column >= j is active
                }
            }
            if (sg[0].n() == 0) { fine = 0; lead = 0; }
            DBG_ADD(12, fine); DBG_ADD(13, lead);
        }
        asm volatile("bar.sync 2, 256;" ::: "memory");
        if (threadIdx.x == 0) {
            unsigned long long sum = 0, mx_tile = 0, mx_chunk = 0;
            for (int c = 0; c <= GINT_MAX_CHUNKS; c++) {
                if (c < GINT_MAX_CHUNKS && c >= nchunk) continue;
                int m = 0, t = 0;
                for (int q = 0; q < 4; q++) { const int v = dbg_load[c][q] + dbg_load[c][q + 4]; m = max(m, v); t += v; }
                if (c == GINT_MAX_CHUNKS) { sum = t; mx_tile = 4ull * m; } else mx_chunk += 4ull * m;
            }
            atomicAdd(&g_dbg[0], sum); atomicAdd(&g_dbg[1], mx_tile); atomicAdd(&g_dbg[2], mx_chunk); atomicAdd(&g_dbg[3], 1ull);
            atomicAdd(&g_dbg[4], (unsigned long long)nchunk);
        }
    }
#endif
    // lane part of every operand address: row lr of the fragment, point lc of the k-step
    unsigned lane_off = smem_addr(&S.phi[0][0][0][0]) + lr * GINT_ROWB + lc * 8;
    asm volatile("" : "+r"(lane_off));
    for (int c = 0; c < nchunk; c++) {
        const int s = c % GINT_STAGES;
        if (c == 64 / GINT_CUBS) {      // the activity words cover 64 list positions: switch to the second half
#pragma unroll
            for (int k = 0; k < GINT_WARP_SEGS; k++) sg[k].W = S.segWhi[warp + GINT_MMA_WARPS * k];
        }
        DBG_T(t_w0);
        mbar_wait(&S.full[s], (c / GINT_STAGES) & 1);
        DBG_T(t_w1);
        DBG_ADD(6, t_w1 - t_w0);
        const unsigned base = lane_off + s * GINT_STAGEB;
#ifndef GINT_DBG_NO_MMA
#pragma unroll
        for (int k = 0; k < GINT_WARP_SEGS; k++) {
            const unsigned bits = stage_steps(sg[k].W, c);
            if (bits) vl_seg_dispatch(sg[k].n(), acc[k], base + sg[k].oa, base + sg[k].ob, bits);
        }
#endif
        __syncwarp();
        if (lane == 0) mbar_arrive(&S.empty[s]);
        DBG_T(t_w2);
        DBG_ADD(7, t_w2 - t_w1);
    }
    DBG_T(t_loop);
    // flush: element (row, col) -> atom pair (a, b), orbitals (oa, ob) -> canonical block (transposed if the canonical
    // key is (b, a)).  Exact zeros (fragments never touched, atoms that do not overlap inside this batch) are skipped.
#pragma unroll
    for (int k = 0; k < GINT_WARP_SEGS; k++) {
        if (sg[k].n() == 0) continue;
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
    DBG_T(t_end);
    DBG_ADD(8, t_end - t_loop);
    DBG_ADD(9, t_end - t_start);
}

// ---------------------------------------------------------------------------------------------------
// gint_rho main kernel (north_star step 3b).  The density blocks Dh_IJ of the tile are stationary DMMA A operands
// (registers): per cubelet X^T = Dh_seg^T Phi_I (8 orbitals of J x 8 points per column fragment) and
// rho_g += sum_j X_jg Phi_J,jg.  Dh = canonical-half, symmetrised density blocks (k_sym_D).
// DMMA column n of X^T <-> point (n >> 1) + 4 (n & 1) of the cubelet, so that the lane's two results (columns 2 lc,
// 2 lc + 1) meet Phi_J at points lc and lc + 4: the same conflict-free 64-bit shared loads as in vlocal.
template <int N>
__device__ __forceinline__ void rho_cols(const double (&d)[GINT_SEG_COLS][2], int j0, double b0, double b1, unsigned pj, double& p0, double& p1) {
    double x[N][2];
#pragma unroll
    for (int j = 0; j < N; j++) { x[j][0] = 0.0; x[j][1] = 0.0; dmma884(x[j], d[j0 + j][0], b0); }
#pragma unroll
    for (int j = 0; j < N; j++) dmma884(x[j], d[j0 + j][1], b1);
    double f0[N], f1[N];
#pragma unroll
    for (int j = 0; j < N; j++) { f0[j] = lds64(pj + (j0 + j) * 8 * GINT_ROWB); f1[j] = lds64(pj + (j0 + j) * 8 * GINT_ROWB + 32); }
#pragma unroll
    for (int j = 0; j < N; j++) { p0 = fma(x[j][0], f0[j], p0); p1 = fma(x[j][1], f1[j], p1); }
}
template <int N>
__device__ __forceinline__ void rho_seg(const double (&d)[GINT_SEG_COLS][2], unsigned pi, unsigned pj, unsigned bits, double (&part)[4][2]) {
    asm volatile("" : "+r"(pi), "+r"(pj));
#pragma unroll
    for (int q = 0; q < 4; q++) {
        if (!((bits >> q) & 1u)) continue;
        const double b0 = lds64(pi + 64 * q), b1 = lds64(pi + 4 * GINT_ROWB + 64 * q);       // Phi_I[8 row + lc (+4)][point pi(lr) of cubelet q]
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
           const unsigned int* __restrict__ coff, int tab_cells, const double* __restrict__ Dh, double* __restrict__ rho) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TileSmem& S = *reinterpret_cast<TileSmem*>(smem_raw);
    {
        TileView tv0;
        tile_setup(g, S, tv0, tile, bstart, bent, atom_pos, atom_spec, sp, crow, ckey, coff, tab, tab_cells, nullptr);
    }
    const int nchunk = S.tv.nchunk;
    if (nchunk == 0) return;
    const int warp = threadIdx.x >> 5;
    if (warp >= GINT_MMA_WARPS) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" :: "n"(GINT_REGS_EVAL_RHO));
        producer_loop<false>(g, S, nchunk, tab, tab_cells, nullptr);
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" :: "n"(GINT_REGS_MMA_RHO));
    const int lane = threadIdx.x & 31, lr = lane >> 2, lc = lane & 3;
    Seg sg[GINT_WARP_SEGS];
    double d[GINT_WARP_SEGS][GINT_SEG_COLS][2];
#pragma unroll
    for (int k = 0; k < GINT_WARP_SEGS; k++) {
        sg[k] = load_seg(S, warp + GINT_MMA_WARPS * k, S.tv.diag);
        load_dseg(S, sg[k], Dh, d[k]);
    }
    const unsigned phi0 = smem_addr(&S.phi[0][0][0][0]);
    unsigned lane_i = phi0 + lc * GINT_ROWB + ((lr >> 1) + 4 * (lr & 1)) * 8;      // Phi_I: row lc of the k-step, point pi(lr)
    unsigned lane_j = phi0 + lr * GINT_ROWB + lc * 8;                              // Phi_J: row lr, point lc (+4)
    asm volatile("" : "+r"(lane_i), "+r"(lane_j));
    for (int c = 0; c < nchunk; c++) {
        const int s = c % GINT_STAGES;
        if (c == 64 / GINT_CUBS) {      // the activity words cover 64 list positions: switch to the second half
#pragma unroll
            for (int k = 0; k < GINT_WARP_SEGS; k++) sg[k].W = S.segWhi[warp + GINT_MMA_WARPS * k];
        }
        double part[4][2];
#pragma unroll
        for (int q = 0; q < 4; q++) { part[q][0] = 0.0; part[q][1] = 0.0; }
        mbar_wait(&S.full[s], (c / GINT_STAGES) & 1);
        unsigned any = 0;
#pragma unroll
        for (int k = 0; k < GINT_WARP_SEGS; k++) {
            const unsigned bits = stage_steps(sg[k].W, c);
            any |= bits;
            if (bits) rho_seg_dispatch(sg[k].n(), d[k], lane_i + s * GINT_STAGEB + sg[k].oa, lane_j + s * GINT_STAGEB + sg[k].ob, bits, part);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&S.empty[s]);
        if (!any) continue;
        // part[q][e]: point lc + 4e of cubelet q, partial over the lane's orbital row lr -> reduce-scatter over lr (lane bits 2..4)
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
        // the lane now owns value t = lr: point lc + 4 (lr & 1) of cubelet lr >> 1
        int gi, gj, gk;
        if (r1 != 0.0 && stage_point(S, c, 8 * (lr >> 1) + lc + 4 * (lr & 1), gi, gj, gk))
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
            c->d_atom_species, c->d_species, c->d_tab, c->d_crow, c->d_ckey, c->d_coff, c->tab_in_smem ? (int)(c->tab_bytes / 16) : 0, V, c->d_cval);
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
        c->d_atom_species, c->d_species, c->d_tab, c->d_crow, c->d_ckey, c->d_coff, c->tab_in_smem ? (int)(c->tab_bytes / 16) : 0, c->d_cval, rho);
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
