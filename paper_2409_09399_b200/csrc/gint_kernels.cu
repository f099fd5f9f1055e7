// gint_kernels.cu -- the per-call hot path (north_star steps 2 and 3), fp64, sm_100a.
//
// Work decomposition.  The mesh is cut into grid batches (default 8x8x16 points) whose neighbouring
// atom images were listed by gint_init, most active first, each with a 128-bit ACTIVITY MASK over the
// batch's 4x4x8 "cubelets" of 2x2x2 mesh points (bit set = some point of the cubelet lies inside the atom's cutoff
// sphere; Fig. 6: everything else is zero padding).  The neighbours of a batch are split into G
// groups of at most 8 atoms / 104 orbitals = 13 FRAGMENTS of 8 orbital rows.
//
// Step 2 (k_eval_phi, the paper's orbital-value kernel): every (batch, atom, active cubelet) is
// evaluated exactly ONCE per call into a "Phi" scratch buffer laid out as the contraction kernels read it: one SLOT
// per (atom group, cubelet on which the group is active) = [orbital row][8 points] doubles.  The scratch holds one
// WAVE of batches (a few GB; re-read through L2 by the tiles that follow immediately).
//
// Step 3 (k_tiles<vlocal | rho>): persistent CTAs, one per SM, pull TILES = (batch, group I, group J), I <= J, from a queue
// in batch order (tiles sharing a group run at the same time on different SMs, so their slots hit L2).  What a tile has to
// know (atom pairs -> canonical blocks, the cubelets on which both groups are active, which warp works on which block of
// fragments on which cubelet) depends on the geometry only: gint_init writes one PLAN per tile (k_plan_fill).  Per CTA:
//   * the issuer warp (12) pops the queue, fetches the next tiles' plans and streams the slots of the tile's cubelets into a
//     shared-memory ring, all with TMA bulk copies (cp.async.bulk, complete_tx on mbarriers); in gint_rho it also reduces
//     the consumers' partial densities in fixed order and adds them to rho once per tile;
//   * 12 consumer warps (setmaxnreg 152) keep the 104 x 104 block of Phi_I^T diag(V dV) Phi_J (gint_vlocal, Eq. 2
//     PAPER.md:66) or of the density blocks D_IJ (gint_rho, Eq. 3) in REGISTERS as DMMA accumulators /
//     stationary operands: the 13 x 13 fragments are cut into BLOCKS of 2 row fragments x 3..4 column fragments, up to
//     three per warp, dealt so that the four SM sub-partitions carry equal numbers of DMMAs.  Per cubelet a block issues
//     mma.sync.m8n8k4.f64 (DMMA.8x8x4) only if one of its rows and one of its columns are active there.
// Only one of each mirror pair of blocks, (A,B,n) / (B,A,-n), is accumulated ("canonical half"); small streaming
// kernels convert between the public pair-list layout and the canonical layout.
#include "gint_internal.h"

typedef unsigned long long u64;
// activity mask over the (at most 128) cubelets of a batch
struct cmask { u64 lo, hi; };
__device__ __forceinline__ cmask operator|(cmask a, cmask b) { return cmask{a.lo | b.lo, a.hi | b.hi}; }
__device__ __forceinline__ cmask operator&(cmask a, cmask b) { return cmask{a.lo & b.lo, a.hi & b.hi}; }
__device__ __forceinline__ cmask& operator|=(cmask& a, cmask b) { a.lo |= b.lo; a.hi |= b.hi; return a; }
__device__ __forceinline__ bool cbit(const cmask& m, int i) { return ((i < 64 ? m.lo >> i : m.hi >> (i - 64)) & 1ull) != 0; }
__device__ __forceinline__ cmask czero() { return cmask{0ull, 0ull}; }
__device__ __forceinline__ int ccount(const cmask& m) { return __popcll(m.lo) + __popcll(m.hi); }
// number of set bits below bit i
__device__ __forceinline__ int crank(const cmask& m, int i) {
    return i < 64 ? __popcll(m.lo & ((1ull << i) - 1ull)) : __popcll(m.lo) + __popcll(m.hi & ((1ull << (i - 64)) - 1ull));
}
// position of the i-th set bit (i < ccount(m))
__device__ __forceinline__ int cselect(const cmask& m, int i) {
    const unsigned w0 = (unsigned)m.lo, w1 = (unsigned)(m.lo >> 32), w2 = (unsigned)m.hi, w3 = (unsigned)(m.hi >> 32);
    const int c0 = __popc(w0), c1 = c0 + __popc(w1), c2 = c1 + __popc(w2);
    const int k = (i >= c0) + (i >= c1) + (i >= c2);
    const unsigned w = k == 0 ? w0 : (k == 1 ? w1 : (k == 2 ? w2 : w3));
    const int skip = k == 0 ? 0 : (k == 1 ? c0 : (k == 2 ? c1 : c2));
    return 32 * k + (int)__fns(w, 0, i - skip + 1);
}
// cubelet id -> first point of the cubelet inside the batch; point p of a cubelet = (px, py, pz) bits
__device__ __forceinline__ void cubelet_point(int cl, int p, int& ix, int& iy, int& iz) {
    ix = 2 * (cl / (4 * GINT_NCZ)) + (p >> 2); iy = 2 * ((cl / GINT_NCZ) & 3) + ((p >> 1) & 1); iz = GINT_CZ * (cl % GINT_NCZ) + (p & 1);
}

#ifndef GINT_DBG_STATS
#define DBG_T(x)
#define DBG_ADD(i, v)
#else
__device__ unsigned long long g_dbg[16];
__device__ unsigned long long g_dbgw[16][8];
#define DBG_T(x) const long long x = clock64()
#define DBG_ADD(i, v) dbg_acc[i] += (unsigned long long)(v)
extern "C" int gint_debug_counters(unsigned long long* out) { return (int)cudaMemcpyFromSymbol(out, g_dbg, sizeof(g_dbg)); }
extern "C" int gint_debug_warp_counters(unsigned long long* out) { return (int)cudaMemcpyFromSymbol(out, g_dbgw, sizeof(g_dbgw)); }
extern "C" int gint_debug_reset() { unsigned long long z[16 * 8] = {0}; cudaMemcpyToSymbol(g_dbgw, z, sizeof(z)); return (int)cudaMemcpyToSymbol(g_dbg, z, 16 * 8); }
#endif

// ---------------------------------------------------------------------------------------------------
// PTX helpers
__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(u64* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(u64* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(smem_addr(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(u64* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(u64* bar, int parity) {
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}"
                 :: "r"(smem_addr(bar)), "r"(parity) : "memory");
}
// the same on 32-bit shared-memory addresses (the hot loops keep them in registers: a generic pointer costs 64-bit arithmetic)
__device__ __forceinline__ void mbar_arrive_s(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait_s(unsigned bar, unsigned parity) {
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}"
                 :: "r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void sts64(unsigned addr, double v) { asm volatile("st.shared.f64 [%0], %1;" :: "r"(addr), "d"(v) : "memory"); }
// TMA bulk copy global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP.S.G)
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, u64* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(dst), "l"(src), "r"(bytes), "r"(smem_addr(bar)) : "memory");
}

// ---------------------------------------------------------------------------------------------------
// Step 2: orbital evaluation, once per (batch, atom, active cubelet).
// phi = R_s(|d|) Y_lm(d/|d|), zero for |d| >= rc (Fig. 6); radial part (reading R5):
// R = a y_i + b y_{i+1} + (a^3-a) z_i + (b^3-b) z_{i+1} from the knot cells {y, z} of the interval, read with 128-bit
// loads from the shared-memory copy of the table when it fits.  A quarter warp = one (atom, cubelet) item, lane = point.
struct EvalSmem {
    double pos[GINT_MAX_NB][4];             // image position, rc^2
    cmask amask[GINT_MAX_NB];
    int tab_off[GINT_MAX_NB], n_int[GINT_MAX_NB], nsh[GINT_MAX_NB], lpack[GINT_MAX_NB];
    int row0[GINT_MAX_NB], norb[GINT_MAX_NB], grp[GINT_MAX_NB];
    int item0[GINT_MAX_NB + 1];             // prefix sums of the atoms' active cubelets
    int zitem0[GINT_MAX_NB + 1];            // prefix sums of the atoms' (group slot) pairs
    int sitem0[GINT_MAX_GROUPS + 1];        // prefix sums of the groups' slots
    cmask gmask[GINT_MAX_GROUPS];
    u64 gbase[GINT_MAX_GROUPS];             // first row of the group's slot array in the wave's Phi scratch
    int gR[GINT_MAX_GROUPS], gfirst[GINT_MAX_GROUPS], gcnt[GINT_MAX_GROUPS], gns[GINT_MAX_GROUPS];
};
#define GINT_EVAL_TAB_OFF ((sizeof(EvalSmem) + 15) & ~(size_t)15)

// gint_vlocal (V != nullptr) stores sqrt(|V dV|) phi: the contraction Phi_I^T diag(V dV) Phi_J then needs no FP64 multiply, only
// the sign of V at the point, which the consumers apply to one operand with an integer XOR (an FP64 multiply queues behind the
// other warps' DMMAs in the shared FP64 pipe).  Points outside the mesh (ragged edge batches) get weight 0.
template <bool TAB_SMEM, bool VL>
__global__ void __launch_bounds__(GINT_EVAL_THREADS)
k_eval_phi(Geom g, long long b0, const int* __restrict__ bstart, const NeighEntry* __restrict__ bent,
           const int* __restrict__ gstart, const u64* __restrict__ goff, u64 wave_row0,
           const double* __restrict__ atom_pos, const int* __restrict__ atom_spec, const SpeciesDev* __restrict__ sp,
           const double* __restrict__ tab, int tab_cells, const double* __restrict__ V, double* __restrict__ phi) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    EvalSmem& S = *reinterpret_cast<EvalSmem*>(smem_raw);
    const long long b = b0 + blockIdx.x;
    const int e0 = bstart[b], n = bstart[b + 1] - e0;
    if (n == 0) return;
    const int tid = threadIdx.x;
    const int G = gstart[b + 1] - gstart[b];
    if (TAB_SMEM) {
        const double2* src = reinterpret_cast<const double2*>(tab);
        double2* dst = reinterpret_cast<double2*>(smem_raw + GINT_EVAL_TAB_OFF);
        for (int i0 = tid; i0 < tab_cells; i0 += 8 * GINT_EVAL_THREADS) {
            double2 tmp[8];
#pragma unroll
            for (int u = 0; u < 8; u++) if (i0 + u * GINT_EVAL_THREADS < tab_cells) tmp[u] = __ldg(src + i0 + u * GINT_EVAL_THREADS);
#pragma unroll
            for (int u = 0; u < 8; u++) if (i0 + u * GINT_EVAL_THREADS < tab_cells) dst[i0 + u * GINT_EVAL_THREADS] = tmp[u];
        }
    }
    const int bz = (int)(b % g.nb[2]), by = (int)((b / g.nb[2]) % g.nb[1]), bx = (int)(b / ((long long)g.nb[2] * g.nb[1]));
    const int i0 = bx * g.bs[0], j0 = by * g.bs[1], k0 = bz * g.bs[2];
    if (tid < n) {
        const NeighEntry e = bent[e0 + tid];
        int t1, t2, t3; unpack_shift(e.shift, t1, t2, t3);
        double x, y, z;
        image_pos(g, atom_pos + 3 * e.atom, t1, t2, t3, x, y, z);
        const SpeciesDev* Sp = sp + atom_spec[e.atom];
        S.pos[tid][0] = x; S.pos[tid][1] = y; S.pos[tid][2] = z; S.pos[tid][3] = Sp->rc * Sp->rc;
        S.amask[tid] = cmask{e.mask[0], e.mask[1]};
        S.tab_off[tid] = Sp->tab_off; S.n_int[tid] = Sp->n_int; S.nsh[tid] = Sp->n_shell; S.norb[tid] = Sp->norb;
        int lp = 0;
        for (int k = 0; k < Sp->n_shell; k++) lp |= Sp->l[k] << (2 * k);
        S.lpack[tid] = lp;
    }
    __syncthreads();
    if (tid < G) {      // one thread per group: entry range, rows, union mask
        const int k = tid, f = group_begin(k, n, G), l = group_begin(k + 1, n, G);
        cmask m = czero();
        int rows = 0;
        for (int e = f; e < l; e++) { m |= S.amask[e]; S.row0[e] = rows; S.grp[e] = k; rows += S.norb[e]; }
        S.gmask[k] = m; S.gfirst[k] = f; S.gcnt[k] = l - f; S.gR[k] = (rows + 7) & ~7; S.gns[k] = ccount(m);
        S.gbase[k] = goff[gstart[b] + k] - wave_row0;
    }
    __syncthreads();
    if (tid == 0) {
        int a = 0, z = 0;
        for (int e = 0; e < n; e++) { S.item0[e] = a; S.zitem0[e] = z; a += ccount(S.amask[e]); z += S.gns[S.grp[e]]; }
        S.item0[n] = a; S.zitem0[n] = z;
        int q = 0;
        for (int k = 0; k < G; k++) { S.sitem0[k] = q; q += S.gns[k]; }
        S.sitem0[G] = q;
    }
    __syncthreads();
    const double2* tb = TAB_SMEM ? reinterpret_cast<const double2*>(smem_raw + GINT_EVAL_TAB_OFF) : reinterpret_cast<const double2*>(tab);
    const int qw = tid >> 3, pl = tid & 7;
    // ---- pass A: the active (atom, cubelet) items, compacted: every quarter warp evaluates one
    const int n_items = S.item0[n];
    for (int it0 = 0; it0 < n_items; it0 += GINT_EVAL_THREADS / 8) {
        const int it = it0 + qw;
        const bool on = it < n_items;
        int e = 0;
        if (on) {       // entry of the item: last e with item0[e] <= it
            int lo = 0, hi = n - 1;
            while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (S.item0[mid] <= it) lo = mid; else hi = mid - 1; }
            e = lo;
        }
        const int k = S.grp[e];
        const int cl = on ? cselect(S.amask[e], it - S.item0[e]) : 0;
        const int slot = crank(S.gmask[k], cl);
        int ix, iy, iz; cubelet_point(cl, pl, ix, iy, iz);
        double px, py, pz;
        mesh_point(g, i0 + ix, j0 + iy, k0 + iz, px, py, pz);
        const double dx = px - S.pos[e][0], dy = py - S.pos[e][1], dz = pz - S.pos[e][2];
        const double rc2 = S.pos[e][3];
        const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
        const bool inside = on && r2 < rc2;
        // 1/r by one Newton step from the single-precision reciprocal square root: relative error 2.4e-7 -> 1.5 e^2 = 9e-14,
        // three orders below the 1e-10 parity bar
        const double q = fmin(fmax(r2, 1e-30), rc2);
        double ir = (double)rsqrtf((float)q);
        ir = ir * fma(-0.5 * q, ir * ir, 1.5);
        const double r = q * ir;
        const int nsh = on ? S.nsh[e] : 0;
        const double x = r * g.inv_dr;
        int i = (int)x;
        i = min(i, S.n_int[e] - 1);
        const double bb = x - (double)i, am = 1.0 - bb;
        const double a3 = (am * am - 1.0) * am, b3 = (bb * bb - 1.0) * bb;
        const double2* row = tb + (S.tab_off[e] + i * nsh);
        const bool tiny = r < 1e-12;
        if (tiny) ir = 0.0;
        // lanes outside the sphere run the same instructions on a clamped radius and store zeros
        double w0 = inside ? 1.0 : 0.0;
        if (VL) {
            const int gi = i0 + ix, gj = j0 + iy, gk = k0 + iz;
            const bool in_mesh = ix < g.bs[0] && iy < g.bs[1] && iz < g.bs[2] && gi < g.N[0] && gj < g.N[1] && gk < g.N[2];    // a point of this batch
            w0 = (inside && in_mesh) ? sqrt(fabs(__ldg(V + ((size_t)gi * g.N[1] + gj) * g.N[2] + gk) * g.dV)) : 0.0;
        }
        const double ux = dx * ir, uy = dy * ir, uz = dz * ir;
        double yw[9];
        {
            const double c1 = 0.4886025119029199 * w0, c2 = (tiny ? 0.0 : 1.0925484305920792) * w0;     // l > 0 orbitals vanish at the nucleus
            const double c20 = (tiny ? 0.0 : 0.31539156525252005) * w0, c22 = (tiny ? 0.0 : 0.5462742152960396) * w0;
            const double c2x = c2 * ux, c2y = c2 * uy;
            yw[0] = 0.28209479177387814 * w0;
            yw[1] = c1 * uy; yw[2] = c1 * uz; yw[3] = c1 * ux;
            yw[4] = c2x * uy; yw[5] = c2y * uz; yw[6] = c20 * fma(3.0 * uz, uz, -1.0); yw[7] = c2x * uz; yw[8] = c22 * fma(ux, ux, -uy * uy);
        }
        // SWIZZLE (gint_rho): point p of slot row r sits at position p ^ (4 * ((r >> 1) & 1)) of the row's 64 bytes.  The B operands of gint_rho
        // (64-bit loads, a half warp = 4 consecutive rows x 4 points) would otherwise hit every bank twice (rows r and r + 2).
        double* o0 = phi + ((S.gbase[k] + (u64)slot * (S.gR[k] + 1) + S.row0[e]) << 3);
        int orow = S.row0[e];
        const int lpack = S.lpack[e];
        const int swz = VL ? 0 : 2;     // gint_rho only (gint_vlocal reads its slots with conflict-free 128-bit loads as they are)
#define GINT_PUT(m) do { o0[pl ^ ((orow & swz) << 1)] = R * yw[m]; o0 += 8; orow++; } while (0)
        for (int s = 0; s < nsh; s++) {
            const double2 c0 = row[s], c1 = row[nsh + s];
            const double R = fma(am, c0.x, fma(bb, c1.x, fma(a3, c0.y, b3 * c1.y)));
            const int l = (lpack >> (2 * s)) & 3;
            if (l == 0) {
                GINT_PUT(0);
            } else if (l == 1) {
                GINT_PUT(1); GINT_PUT(2); GINT_PUT(3);
            } else {
                GINT_PUT(4); GINT_PUT(5); GINT_PUT(6); GINT_PUT(7); GINT_PUT(8);
            }
        }
#undef GINT_PUT
    }
    // ---- pass B: zero rows.  The contraction kernels read a slot in blocks of fragments and only test whether SOME row and SOME
    // column fragment of a block is active on the cubelet: every row of a slot that no active atom owns (inactive atoms, the padding
    // rows behind the group's last orbital) must hold zeros.
    const int n_z = S.zitem0[n];
    for (int it = qw; it < n_z; it += GINT_EVAL_THREADS / 8) {
        int lo = 0, hi = n - 1;
        while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (S.zitem0[mid] <= it) lo = mid; else hi = mid - 1; }
        const int e = lo, k = S.grp[e], slot = it - S.zitem0[e];
        const int cl = cselect(S.gmask[k], slot);
        const bool act = cbit(S.amask[e], cl);
        const bool last = e == S.gfirst[k] + S.gcnt[k] - 1;
        int r0 = S.row0[e], r1 = r0 + S.norb[e];
        if (act) r0 = r1;                               // an active atom's own rows were written by pass A
        if (last) r1 = S.gR[k];                         // padding rows
        double* o0 = phi + ((S.gbase[k] + (u64)slot * (S.gR[k] + 1)) << 3) + pl;
        for (int rr = r0; rr < r1; rr++) o0[rr << 3] = 0.0;
    }
    // ---- pass C (gint_vlocal): the sign row of every slot: -0.0 where V < 0 at the point, else +0.0
    if (VL) {
        const int n_s = S.sitem0[G];
        for (int it = qw; it < n_s; it += GINT_EVAL_THREADS / 8) {
            int k = 0;
            while (S.sitem0[k + 1] <= it) k++;
            const int slot = it - S.sitem0[k];
            const int cl = cselect(S.gmask[k], slot);
            int ix, iy, iz; cubelet_point(cl, pl, ix, iy, iz);
            const int gi = i0 + ix, gj = j0 + iy, gk = k0 + iz;
            const bool in_batch = ix < g.bs[0] && iy < g.bs[1] && iz < g.bs[2] && gi < g.N[0] && gj < g.N[1] && gk < g.N[2];
            const bool neg = in_batch && __ldg(V + ((size_t)gi * g.N[1] + gj) * g.N[2] + gk) < 0.0;
            phi[((S.gbase[k] + (u64)slot * (S.gR[k] + 1) + S.gR[k]) << 3) + pl] = neg ? -0.0 : 0.0;
        }
    }
}


// ---------------------------------------------------------------------------------------------------
// Tile plans (gint_init).  k_plan_count: plan size of every tile (one thread per tile); k_plan_fill: one CTA per tile.
__global__ void __launch_bounds__(256) k_plan_count(long long n_tiles, const int2* __restrict__ tile, const int* __restrict__ bstart,
                                                    const NeighEntry* __restrict__ bent, int* __restrict__ units) {
    const long long ti = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (ti >= n_tiles) return;
    const int2 td = tile[ti];
    const int b = td.x, I = td.y & 255, J = (td.y >> 8) & 255, G = (td.y >> 16) & 255;
    const int e0 = bstart[b], n = bstart[b + 1] - e0;
    cmask mI = czero(), mJ = czero();
    for (int e = group_begin(I, n, G); e < group_begin(I + 1, n, G); e++) { const NeighEntry en = bent[e0 + e]; mI |= cmask{en.mask[0], en.mask[1]}; }
    for (int e = group_begin(J, n, G); e < group_begin(J + 1, n, G); e++) { const NeighEntry en = bent[e0 + e]; mJ |= cmask{en.mask[0], en.mask[1]}; }
    units[ti] = (int)plan_units(ccount(mI & mJ));
}

struct PlanScratch {
    cmask amask[16];                    // slot s < 8: atom s of group I; slot 8 + s: atom s of group J
    cmask fmask[2][16];                 // [side][fragment]: OR of amask over the atoms with orbitals in the fragment
    int atom[16], shift[16];
    int cstart[2][GINT_TILE_ATOMS + 1]; // first orbital row of each atom inside its group
    unsigned cubinfo[GINT_NCUB];        // per listed cubelet: active row fragments of I | active column fragments of J << 16
    unsigned char asc[GINT_NCUB];       // the cubelets on which both groups are active, ascending
    int stride;
};
struct alignas(16) PlanSmem {
    PlanHdr H;
    PlanCub C[GINT_NCUB + GINT_SC + 1];
    PlanScratch Q;
};
#ifdef GINT_DBG_STATS
__device__ unsigned long long g_plan_stats[16];
extern "C" int gint_debug_plan_stats(unsigned long long* out) { return (int)cudaMemcpyFromSymbol(out, g_plan_stats, sizeof(g_plan_stats)); }
#endif

__global__ void __launch_bounds__(GINT_PLAN_THREADS)
k_plan_fill(Geom g, const int2* __restrict__ tile, const int* __restrict__ bstart, const NeighEntry* __restrict__ bent,
            const int* __restrict__ gstart, const u64* __restrict__ goff, const int* __restrict__ atom_spec,
            const SpeciesDev* __restrict__ sp, const int* __restrict__ crow, const u64* __restrict__ ckey,
            const unsigned int* __restrict__ coff, const unsigned* __restrict__ planoff, unsigned char* __restrict__ plan) {
    __shared__ PlanSmem P;
    PlanHdr& X = P.H;
    PlanScratch& Q = P.Q;
    const int sid = threadIdx.x, lane = sid & 31, sw = sid >> 5;
    const int2 td = tile[blockIdx.x];
    const int b = td.x, I = td.y & 255, J = (td.y >> 8) & 255, G = (td.y >> 16) & 255;
    const bool diag = I == J;
    const int e0 = bstart[b], n = bstart[b + 1] - e0;
    const int eI = group_begin(I, n, G), eJ = group_begin(J, n, G);
    const int nI = group_begin(I + 1, n, G) - eI, nJ = group_begin(J + 1, n, G) - eJ;
    {   // the records are copied out whole: no stale bytes
        unsigned* z = reinterpret_cast<unsigned*>(P.C);
        for (int i = sid; i < (int)(sizeof(P.C) / 4); i += GINT_PLAN_THREADS) z[i] = 0u;
    }
    if (sid < 16) {
        const int side = sid >> 3, a = sid & 7;
        const bool valid = a < (side ? nJ : nI);
        int atom = 0, shift = pack_shift(0, 0, 0), norb = 0;
        cmask m = czero();
        if (valid) {
            const NeighEntry e = bent[e0 + (side ? eJ : eI) + a];
            atom = e.atom; shift = e.shift; m = cmask{e.mask[0], e.mask[1]};
            norb = sp[atom_spec[atom]].norb;
        }
        Q.atom[sid] = atom; Q.shift[sid] = shift; Q.amask[sid] = m;
        int inc = norb;
#pragma unroll
        for (int dlt = 1; dlt < 8; dlt <<= 1) { const int t = __shfl_up_sync(0xffffu, inc, dlt, 8); if (a >= dlt) inc += t; }
        Q.cstart[side][a] = inc - norb;
        if (a == 7) Q.cstart[side][8] = inc;
    }
    __syncthreads();
    const int totI = Q.cstart[0][GINT_TILE_ATOMS], totJ = Q.cstart[1][GINT_TILE_ATOMS];
    const int nfI = (totI + 7) >> 3, nfJ = (totJ + 7) >> 3;
    if (sid < 64) {
        // canonical block of every atom pair of the tile: binary search in row A of the canonical key list
        const int a = sid >> 3, bb = sid & 7;
        PairEnt pe; pe.off = 0xffffffffu; pe.sr = 0; pe.sc = 0;
        // diagonal tile: only pairs a <= b are accumulated (a == b is the full on-site block)
        if (a < nI && bb < nJ && !(diag && a > bb)) {
            int A = Q.atom[a], B = Q.atom[8 + bb];
            const int nA = Q.cstart[0][a + 1] - Q.cstart[0][a], nB = Q.cstart[1][bb + 1] - Q.cstart[1][bb];
            int ta1, ta2, ta3, tb1, tb2, tb3;
            unpack_shift(Q.shift[a], ta1, ta2, ta3); unpack_shift(Q.shift[8 + bb], tb1, tb2, tb3);
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
        X.pair[a][bb] = pe;
    } else {
        // fragment masks, then the row maps
        const int q = sid - 64, side = q >> 4, f = q & 15;
        cmask fm = czero();
        for (int k = 0; k < GINT_TILE_ATOMS; k++)
            if (Q.cstart[side][k] < 8 * f + 8 && Q.cstart[side][k + 1] > 8 * f) fm |= Q.amask[8 * side + k];
        Q.fmask[side][f] = fm;
        for (int idx = q; idx < 2 * GINT_TILE_ORB; idx += 32) {
            const int sd = idx / GINT_TILE_ORB, row = idx - sd * GINT_TILE_ORB;
            int a = 255, o = 0;
            for (int k = 0; k < GINT_TILE_ATOMS; k++)
                if (row >= Q.cstart[sd][k] && row < Q.cstart[sd][k + 1]) { a = k; o = row - Q.cstart[sd][k]; }
            X.row_atom[sd][row] = (unsigned char)a; X.row_orb[sd][row] = (unsigned char)o;
        }
    }
    __syncthreads();
    cmask mI = czero(), mJ = czero();       // union masks of the two groups (every thread)
#pragma unroll
    for (int a = 0; a < 8; a++) { mI |= Q.amask[a]; mJ |= Q.amask[8 + a]; }
    const cmask U = mI & mJ;
    const int ncub = ccount(U);
    if (sw == 0) {
        // the cubelets on which both groups are active, ascending
        const unsigned Uw[4] = {(unsigned)U.lo, (unsigned)(U.lo >> 32), (unsigned)U.hi, (unsigned)(U.hi >> 32)};
        const unsigned lt = (1u << lane) - 1u;
        int before = 0;
#pragma unroll
        for (int wd = 0; wd < 4; wd++) {
            if ((Uw[wd] >> lane) & 1u) Q.asc[before + __popc(Uw[wd] & lt)] = (unsigned char)(32 * wd + lane);
            before += __popc(Uw[wd]);
        }
    } else if (sid == 32) {
        const int bz = b % g.nb[2], by = (b / g.nb[2]) % g.nb[1], bx = b / (g.nb[2] * g.nb[1]);
        X.i0 = bx * g.bs[0]; X.j0 = by * g.bs[1]; X.k0 = bz * g.bs[2];
        X.ex = min(g.bs[0], g.N[0] - X.i0); X.ey = min(g.bs[1], g.N[1] - X.j0); X.ez = min(g.bs[2], g.N[2] - X.k0);
        X.nI = nI; X.nJ = nJ; X.nfI = nfI; X.nfJ = nfJ; X.RI = 8 * nfI; X.RJ = 8 * nfJ; X.diag = diag;
        X.pad0 = X.pad1 = X.pad2 = 0;
        X.rowI = goff[gstart[b] + I]; X.rowJ = goff[gstart[b] + J];
        X.valid = 1; X.zero = 0; X.ncub = ncub; X.nstage = (ncub + GINT_SC - 1) / GINT_SC;
        // A ring stage holds two neighbours of the ascending list (mostly neighbours along a3: similar activity, gint_rho visits a
        // stage as a whole).  The pairs are walked with a stride coprime to their number (about 0.62 of it): any window of a few
        // consecutive stages then samples the whole batch, so the work of the consumer warps (whose blocks are active on different
        // parts of the batch) stays balanced inside the few ring stages they may drift apart.  An odd last cubelet comes last.
        int s = 1;
#ifndef GINT_PLAN_NO_SCRAMBLE
        const int npair = ncub / GINT_SC;
        if (npair > 2) {
            s = max(1, (npair * 618) / 1000);
            for (;; s++) { int x = s, y = npair; while (y) { const int t = x % y; x = y; y = t; } if (x == 1) break; }
        }
#endif
        Q.stride = s;
    } else if (sid == 64) {
        // Block plan.  The 13 x 13 fragments of the tile are cut into blocks of two adjacent row fragments x 3 or 4 adjacent column
        // fragments (neighbours are sorted by falling activity, so the fragments of a block have similar activity masks).  A block is
        // worked on a cubelet iff one of its rows and one of its columns are active there; its cost = 4 n DMMAs per such cubelet.
        // In a diagonal tile only blocks that reach the atom diagonal or lie above it exist.  Blocks are dealt heaviest first to the
        // least loaded SM sub-partition (consumer warp w runs on sub-partition w % 4) and there to the least loaded warp with a free slot.
        for (int k = 0; k < GINT_WARP_BLOCKS; k++) for (int w = 0; w < GINT_MMA_WARPS; w++) X.blk[k][w] = 0;
        unsigned desc[28];
        int wgt[28], np = 0;
        // column groups of 3 fragments; one group of 4 (the first: the densest columns) when 3 does not divide evenly, else a last group of 2
        const int ng = nfJ <= 4 ? 1 : (nfJ + 2) / 3 - (nfJ % 3 == 1);
        for (int r0 = 0; r0 < nfI; r0 += 2) {
            const bool has1 = r0 + 1 < nfI;
            const int cf0 = diag ? (Q.cstart[1][X.row_atom[0][8 * r0]] >> 3) : 0;
            const cmask rm = has1 ? (Q.fmask[0][r0] | Q.fmask[0][r0 + 1]) : Q.fmask[0][r0];
            int c0 = 0;
            for (int gi = 0; gi < ng; gi++) {
                const int nn = ng == 1 ? nfJ : ((gi == 0 && nfJ % 3 == 1) ? 4 : min(3, nfJ - c0));
                if (c0 + nn > cf0) {                    // the block holds a fragment on or above the diagonal
                    cmask cm = czero();
                    for (int j = 0; j < nn; j++) cm |= Q.fmask[1][c0 + j];
                    desc[np] = (unsigned)r0 | ((unsigned)has1 << 4) | ((unsigned)c0 << 5) | ((unsigned)nn << 9);
                    wgt[np] = ccount(rm & cm) * nn * (has1 ? 2 : 1);
                    np++;
                }
                c0 += nn;
            }
        }
        for (int i = 1; i < np; i++) {      // insertion sort by falling weight
            const unsigned d = desc[i]; const int w = wgt[i];
            int j = i - 1;
            while (j >= 0 && wgt[j] < w) { desc[j + 1] = desc[j]; wgt[j + 1] = wgt[j]; j--; }
            desc[j + 1] = d; wgt[j + 1] = w;
        }
        int lsm[4] = {0, 0, 0, 0}, lw[GINT_MMA_WARPS], used[GINT_MMA_WARPS];
        for (int w = 0; w < GINT_MMA_WARPS; w++) { lw[w] = 0; used[w] = 0; }      // used: bit k = block slot k taken
        for (int pass = 0; pass < 2; pass++)            // the 4-column blocks first: only block slot 0 holds them (at most 7 of them, 12 slots)
            for (int i = 0; i < np; i++) {
                const bool wide = ((desc[i] >> 9) & 15u) > 3;
                if (wide != (pass == 0)) continue;
                int best = -1;
                for (int w = 0; w < GINT_MMA_WARPS; w++) {
                    const bool free_slot = wide ? !(used[w] & 1) : used[w] != (1 << GINT_WARP_BLOCKS) - 1;
                    if (!free_slot) continue;
                    if (best < 0 || lsm[w & 3] < lsm[best & 3] || (lsm[w & 3] == lsm[best & 3] && lw[w] < lw[best])) best = w;
                }
                if (best < 0) __trap();     // cannot happen: at most 28 blocks (7 of them wide) for GINT_WARP_BLOCKS * GINT_MMA_WARPS slots
                int k = 0;
                if (!wide) {                // a narrow block prefers the slots that cannot hold a wide one
                    k = 0;
                    for (int kk = GINT_WARP_BLOCKS - 1; kk >= 1; kk--) if (!(used[best] & (1 << kk))) k = kk;
                }
                used[best] |= 1 << k; lsm[best & 3] += wgt[i]; lw[best] += wgt[i];
                X.blk[k][best] = desc[i];
            }
    }
    __syncthreads();
    // the listed cubelets in walking order, their slots and which fragments are active there
    for (int pos = sid; pos < ncub; pos += GINT_PLAN_THREADS) {
        const int npair = ncub / GINT_SC;
        const int cl = pos < GINT_SC * npair ? Q.asc[GINT_SC * (int)(((long long)(pos / GINT_SC) * Q.stride) % npair) + pos % GINT_SC] : Q.asc[pos];
        PlanCub& c = P.C[pos];
        c.cub = (unsigned char)cl;
        c.slotI = (unsigned short)crank(mI, cl); c.slotJ = (unsigned short)crank(mJ, cl);
        unsigned info = 0;
        for (int f = 0; f < nfI; f++) info |= (unsigned)cbit(Q.fmask[0][f], cl) << f;
        for (int f = 0; f < nfJ; f++) info |= (unsigned)cbit(Q.fmask[1][f], cl) << (16 + f);
        Q.cubinfo[pos] = info;
    }
    __syncthreads();
    // visit codes: which rows of which block every consumer warp works on, per listed cubelet
    for (int idx = sid; idx < ncub * GINT_MMA_WARPS; idx += GINT_PLAN_THREADS) {
        const int pos = idx / GINT_MMA_WARPS, w = idx - pos * GINT_MMA_WARPS;
        const unsigned info = Q.cubinfo[pos];
        unsigned code = 0;
#pragma unroll
        for (int k = 0; k < GINT_WARP_BLOCKS; k++) {
            const unsigned d = X.blk[k][w];
            const unsigned rr = (info >> (d & 15u)) & (((d >> 4) & 1u) ? 3u : 1u);
            const unsigned cm = (info >> (16 + ((d >> 5) & 15u))) & ((1u << ((d >> 9) & 7u)) - 1u);
#ifdef GINT_DBG_DENSE
            if ((d >> 9) & 7u) code |= (((d >> 4) & 1u) ? 3u : 1u) << (2 * k);
#else
            if (cm) code |= rr << (2 * k);
#endif
        }
        P.C[pos].vis[w] = (unsigned char)code;
    }
    __syncthreads();
#ifdef GINT_DBG_STATS
    if (sid == 1) {
        // DMMAs per tile at several granularities of skipping (debug statistics)
        unsigned long long fine = 0, atomx = 0, dense = 0, exec = 0;
        for (int r = 0; r < nfI; r++) {
            const int cf = diag ? (Q.cstart[1][X.row_atom[0][8 * r]] >> 3) : 0;
            for (int cc = cf; cc < nfJ; cc++) fine += 2ull * ccount(Q.fmask[0][r] & Q.fmask[1][cc]);
            dense += 2ull * (nfJ - cf) * ncub;
        }
        for (int a = 0; a < nI; a++) for (int bb = (diag ? a : 0); bb < nJ; bb++) {
            const unsigned long long na = Q.cstart[0][a + 1] - Q.cstart[0][a], nb2 = Q.cstart[1][bb + 1] - Q.cstart[1][bb];
            const unsigned long long el = (diag && a == bb) ? na * (na + 1) / 2 : na * nb2;       // orbital pairs
            atomx += el * ccount(Q.amask[a] & Q.amask[8 + bb]);                                     // x cubelets (8 points each)
        }
        for (int pos = 0; pos < ncub; pos++) for (int w = 0; w < GINT_MMA_WARPS; w++) for (int k = 0; k < GINT_WARP_BLOCKS; k++) {
            const unsigned rr = (P.C[pos].vis[w] >> (2 * k)) & 3u;
            if (rr) exec += (rr == 3u ? 4ull : 2ull) * ((X.blk[k][w] >> 9) & 7u);
        }
        // what-if: a visit covers GR consecutive cubelets of the ascending list (rows / columns active on any of them)
        unsigned long long execg[2] = {0, 0}, visg[3] = {0, 0, 0};
        for (int gi = 0; gi < 3; gi++) {
            const int GR = gi == 0 ? 1 : (gi == 1 ? 2 : 4);
            for (int p0 = 0; p0 < ncub; p0 += GR) {
                unsigned info = 0; int cnt = 0;
                for (int u = 0; u < GR && p0 + u < ncub; u++) {
                    const int cl = Q.asc[p0 + u]; cnt++;
                    for (int f = 0; f < nfI; f++) info |= (unsigned)cbit(Q.fmask[0][f], cl) << f;
                    for (int f = 0; f < nfJ; f++) info |= (unsigned)cbit(Q.fmask[1][f], cl) << (16 + f);
                }
                for (int w = 0; w < GINT_MMA_WARPS; w++) for (int k = 0; k < GINT_WARP_BLOCKS; k++) {
                    const unsigned d = X.blk[k][w];
                    if (!((d >> 9) & 7u)) continue;
                    const unsigned rr = (info >> (d & 15u)) & (((d >> 4) & 1u) ? 3u : 1u);
                    const unsigned cm = (info >> (16 + ((d >> 5) & 15u))) & ((1u << ((d >> 9) & 7u)) - 1u);
                    if (rr && cm) { visg[gi]++; if (gi) execg[gi - 1] += (rr == 3u ? 4ull : 2ull) * ((d >> 9) & 7u) * cnt; }
                }
            }
        }
        // balance of the four SM sub-partitions (consumer warp w runs on w % 4): per window of GINT_NS stages, max / mean of their DMMA counts
        {
            unsigned long long sum_max = 0, sum_all = 0, tot[4] = {0, 0, 0, 0}, win[4] = {0, 0, 0, 0};
            for (int pos = 0; pos < ncub; pos++) {
                for (int w = 0; w < GINT_MMA_WARPS; w++) for (int k = 0; k < GINT_WARP_BLOCKS; k++) {
                    const unsigned rr = (P.C[pos].vis[w] >> (2 * k)) & 3u;
                    if (rr) { const unsigned long long v = (rr == 3u ? 4ull : 2ull) * ((X.blk[k][w] >> 9) & 7u); win[w & 3] += v; tot[w & 3] += v; }
                }
                if ((pos + 1) % (GINT_NS * GINT_SC) == 0 || pos == ncub - 1) {
                    unsigned long long m = 0;
                    for (int q4 = 0; q4 < 4; q4++) { m = win[q4] > m ? win[q4] : m; sum_all += win[q4]; win[q4] = 0; }
                    sum_max += 4 * m;
                }
            }
            unsigned long long mt = 0;
            for (int q4 = 0; q4 < 4; q4++) mt = tot[q4] > mt ? tot[q4] : mt;
            atomicAdd(&g_plan_stats[11], sum_max); atomicAdd(&g_plan_stats[12], sum_all); atomicAdd(&g_plan_stats[13], 4 * mt);
        }
        atomicAdd(&g_plan_stats[6], execg[0]); atomicAdd(&g_plan_stats[7], execg[1]);
        atomicAdd(&g_plan_stats[8], visg[0]); atomicAdd(&g_plan_stats[9], visg[1]); atomicAdd(&g_plan_stats[10], visg[2]);
        atomicAdd(&g_plan_stats[0], fine); atomicAdd(&g_plan_stats[1], atomx); atomicAdd(&g_plan_stats[2], dense); atomicAdd(&g_plan_stats[3], exec);
        atomicAdd(&g_plan_stats[4], (unsigned long long)ncub); atomicAdd(&g_plan_stats[5], 1ull);
    }
#endif
    // copy out
    const unsigned o0 = planoff[blockIdx.x], o1 = planoff[blockIdx.x + 1];
    const uint4* src = reinterpret_cast<const uint4*>(&P);
    uint4* dst = reinterpret_cast<uint4*>(plan + (size_t)o0 * 16);
    for (unsigned i = sid; i < o1 - o0; i += GINT_PLAN_THREADS) dst[i] = src[i];
}

// ---------------------------------------------------------------------------------------------------
// shared memory of the contraction kernels
static_assert(GINT_SC == 2, "the density reduction of the consumers is written for two cubelets per stage");
// gint_rho runs a ring of GINT_NS - 1 stages; the memory of the last stage holds GINT_NRED buffers of the consumers' LANE partial
// densities of a stage, [consumer warp][lane][cubelet of the stage, point 2 (lane % 4) + e] (partial over the lane's orbital row):
// the sum over the 8 rows of a fragment and over the warps is taken by the reducer warps (13, 14) of the issuer's warp group, which
// also add the stage's 16 densities to rho -- the consumers' stage ends with two stores behind its last DMMAs.
#define GINT_NRED 2                 // reducer warps
#ifndef GINT_NBUF
#define GINT_NBUF 4                 // buffers of lane partial densities (a consumer may run this many stages ahead of the reducers)
#endif
#define GINT_LPART_BYTES (GINT_MMA_WARPS * 32 * GINT_SC * 2 * 8)
#define GINT_RHO_RSV ((GINT_NBUF * GINT_LPART_BYTES + GINT_STAGE_BYTES - 1) / GINT_STAGE_BYTES)     // ring stages given up for them
static_assert(GINT_NBUF % GINT_NRED == 0, "a buffer always goes to the same reducer");
struct alignas(128) TileSmem {
    unsigned char ring[GINT_NS][GINT_STAGE_BYTES];     // stage: [cubelet q][side][row][8 points]
    alignas(16) unsigned char plan[GINT_NCTX][GINT_PLAN_MAX_BYTES];    // PlanHdr + PlanCub[]
    u64 full[GINT_NS], empty[GINT_NS];             // stage filled by TMA / read by all consumer warps
    u64 ctx_full[GINT_NCTX], ctx_free[GINT_NCTX];  // plan arrived / released by consumers, issuer and (gint_rho) reducers
    u64 lfull[GINT_NBUF], lempty[GINT_NBUF];       // gint_rho: a buffer of lane partial densities written by all consumers / read by its reducer
};
__device__ __forceinline__ const PlanHdr& plan_hdr(const TileSmem& S, int c) { return *reinterpret_cast<const PlanHdr*>(S.plan[c]); }
__device__ __forceinline__ const PlanCub* plan_cub(const TileSmem& S, int c) { return reinterpret_cast<const PlanCub*>(S.plan[c] + sizeof(PlanHdr)); }

size_t gint_smem_needed(gint_ctx* c, size_t limit) {
    c->tab_in_smem = GINT_EVAL_TAB_OFF + c->tab_bytes <= 72 * 1024 && GINT_EVAL_TAB_OFF + c->tab_bytes <= limit;   // three evaluation CTAs per SM
    c->smem_eval = GINT_EVAL_TAB_OFF + (c->tab_in_smem ? c->tab_bytes : 0);
    return sizeof(TileSmem) + 128;
}

// ---------------------------------------------------------------------------------------------------
// Issuer warp: pops the tile queue, fetches plans, streams the tile's slots into the ring (NSK stages).
template <int NSK>
__device__ __forceinline__ void retire_stage(TileSmem& S, int gr) {
    mbar_wait(&S.empty[gr % NSK], (gr / NSK) & 1);
}

// Reducer warp `id` of gint_rho (stages id, id + GINT_NRED, ... of the CTA's stage sequence): sums the lane partial densities of a
// stage in fixed order and adds the 16 densities to rho (every listed cubelet belongs to exactly one stage of its tile: one
// red.global.add.f64 per mesh point per tile).
__device__ __forceinline__ void reducer_role(const Geom& g, TileSmem& S, int id, double* __restrict__ rho) {
    const int lane = threadIdx.x & 31;
    const int pt = lane & 15, half = lane >> 4, q = pt >> 3, p = pt & 7;
    // lane partial (warp w, lane 4 lr + lc)[2 q + e] with lc = p / 2, e = p % 2
    const double* lp0 = reinterpret_cast<const double*>(&S.ring[GINT_NS - GINT_RHO_RSV][0]) + (size_t)(p >> 1) * 4 + 2 * q + (p & 1);
    int g0 = 0;
    for (int t = 0;; t++) {
        const int c = t % GINT_NCTX;
        mbar_wait(&S.ctx_full[c], (t / GINT_NCTX) & 1);
        const PlanHdr& X = plan_hdr(S, c);
        if (!X.valid) break;
        const PlanCub* C = plan_cub(S, c);
        const int nstage = X.nstage;
        for (int st = 0; st < nstage; st++) {
            const int gs = g0 + st;
            if (gs % GINT_NRED != id) continue;
            const int lb = gs % GINT_NBUF;
            const double* lp = lp0 + (size_t)lb * (GINT_LPART_BYTES / 8);
            mbar_wait(&S.lfull[lb], (gs / GINT_NBUF) & 1);
            double v[4] = {0.0, 0.0, 0.0, 0.0};         // four chains: the adds queue behind the consumers' DMMAs in the FP64 pipe
#pragma unroll
            for (int w = 0; w < GINT_MMA_WARPS / 2; w++)
#pragma unroll
                for (int lr = 0; lr < 8; lr++) v[lr & 3] += lp[((size_t)(half * (GINT_MMA_WARPS / 2) + w) * 32 + lr * 4) * 4];
            double sum = (v[0] + v[1]) + (v[2] + v[3]);
            sum += __shfl_xor_sync(0xffffffffu, sum, 16);
            __syncwarp();
            if (lane == 0) mbar_arrive(&S.lempty[lb]);
            const int ncs = min(GINT_SC, X.ncub - st * GINT_SC);
            if (half == 0 && q < ncs) {
                int ix, iy, iz; cubelet_point(C[st * GINT_SC + q].cub, p, ix, iy, iz);
                if (sum != 0.0 && ix < X.ex && iy < X.ey && iz < X.ez)
                    atomicAdd(rho + ((size_t)(X.i0 + ix) * g.N[1] + (X.j0 + iy)) * g.N[2] + (X.k0 + iz), sum);
            }
        }
        g0 += nstage;
        __syncwarp();
        if (lane == 0) mbar_arrive(&S.ctx_free[c]);
    }
}

template <bool VLOCAL>
__device__ __forceinline__ void issuer_role(const Geom& g, TileSmem& S, const unsigned char* __restrict__ plan, const unsigned* __restrict__ planoff,
                                            int n_tiles, int* __restrict__ queue, const double* __restrict__ phi, u64 wave_row0, double* __restrict__ rho) {
    const int lane = threadIdx.x & 31;
    constexpr int NSK = VLOCAL ? GINT_NS : GINT_NS - GINT_RHO_RSV;     // gint_rho: the last stages' memory holds the lane partial densities
    int gi = 0, gr = 0;                 // stages issued / retired
    int requested = 0;                  // plans requested so far
    bool drained = false;               // the queue has run out
    // request the plan of the next tile into context requested % GINT_NCTX
    auto request = [&]() {
        const int t = requested, c = t % GINT_NCTX;
        if (t >= GINT_NCTX) {
            // the context's previous tile must be over: consumers, issuer (and the reducers of gint_rho) have left it
            mbar_wait(&S.ctx_free[c], ((t / GINT_NCTX) - 1) & 1);
        }
        int ti = 0;
        if (lane == 0) ti = atomicAdd(queue, 1);
        ti = __shfl_sync(0xffffffffu, ti, 0);
        if (ti >= n_tiles) {
            if (lane == 0) {
                reinterpret_cast<PlanHdr*>(S.plan[c])->valid = 0;              // a generic store into a buffer the bulk copies also write
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                mbar_arrive(&S.ctx_full[c]);
            }
            drained = true;
        } else if (lane == 0) {
            const unsigned o0 = __ldg(planoff + ti), o1 = __ldg(planoff + ti + 1);
            mbar_expect_tx(&S.ctx_full[c], (o1 - o0) * 16u);
            bulk_g2s(smem_addr(S.plan[c]), plan + (size_t)o0 * 16, (o1 - o0) * 16u, &S.ctx_full[c]);
        }
        requested++;
    };
    for (int k = 0; k < GINT_NCTX - 2 && !drained; k++) request();
    for (int t = 0;; t++) {
        const int c = t % GINT_NCTX;
        if (!drained && requested < t + GINT_NCTX - 1) request();    // into the context of tile t - 2, which the consumers have left or are about to (tile t - 1 still has stages in the ring)
        mbar_wait(&S.ctx_full[c], (t / GINT_NCTX) & 1);
        const PlanHdr& X = plan_hdr(S, c);
        if (!X.valid) break;
        const PlanCub* C = plan_cub(S, c);
        const int nstage = X.nstage, ncub = X.ncub;
        const unsigned strI = (unsigned)(X.RI + 1) * GINT_ROW_BYTES, strJ = (unsigned)(X.RJ + 1) * GINT_ROW_BYTES;     // slot strides
        const unsigned bI = VLOCAL ? strI : strI - GINT_ROW_BYTES;                 // gint_vlocal also needs the sign row of side I
        const unsigned bJ = X.diag ? 0u : strJ - GINT_ROW_BYTES;
        const unsigned char* srcI = reinterpret_cast<const unsigned char*>(phi) + (X.rowI - wave_row0) * GINT_ROW_BYTES;
        const unsigned char* srcJ = reinterpret_cast<const unsigned char*>(phi) + (X.rowJ - wave_row0) * GINT_ROW_BYTES;
        for (int st = 0; st < nstage; st++, gi++) {
            const int s = gi % NSK;
            while (gi - gr >= NSK) { retire_stage<NSK>(S, gr); gr++; }
            const int ncs = min(GINT_SC, ncub - st * GINT_SC);
#ifdef GINT_DBG_NO_TMA
            if (lane == 0) mbar_arrive(&S.full[s]);
            __syncwarp();
            if (false) {
#else
            if (lane == 0) mbar_expect_tx(&S.full[s], (unsigned)ncs * (bI + bJ));
            __syncwarp();
            if (lane < ncs) {
#endif
                const PlanCub& pc = C[st * GINT_SC + lane];
                const unsigned dst = smem_addr(&S.ring[s][lane * 2 * GINT_SLOT_MAX_BYTES]);
                bulk_g2s(dst, srcI + (size_t)pc.slotI * strI, bI, &S.full[s]);
                if (bJ) bulk_g2s(dst + GINT_SLOT_MAX_BYTES, srcJ + (size_t)pc.slotJ * strJ, bJ, &S.full[s]);
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&S.ctx_free[c]);          // the issuer is done with the plan
    }
    while (gr < gi) { retire_stage<NSK>(S, gr); gr++; }
}

// ---------------------------------------------------------------------------------------------------
// ---------------------------------------------------------------------------------------------------
// Consumers.  DMMA.8x8x4 fragment layouts (mma.sync.m8n8k4.f64): A[m = lane / 4][k = lane % 4], B[k = lane % 4][n = lane / 4],
// C[m = lane / 4][n = 2 (lane % 4) + {0, 1}].  A slot row holds the 8 points of a cubelet; the two k-steps of a cubelet
// take points {0,2,4,6} and {1,3,5,7}, so that one 128-bit load fetches a lane's operands of both steps.
__device__ __forceinline__ double2 lds128(unsigned addr) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ unsigned lds_u8(unsigned addr) {
    unsigned v;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ double lds64(unsigned addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr) : "memory");
    return v;
}
#define GINT_DMMA(c0, c1, a, b) "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {" c0 "," c1 "},{" a "},{" b "},{" c0 "," c1 "};\n\t"
// A DMMA that is predicated off still occupies the FP64 tensor pipe for its 16 cycles (measured), and ptxas turns a
// forward branch over a few DMMAs into predication.  So every skippable DMMA sequence is written as a loop with an opaque,
// never-taken back edge (q == 0 at run time): ptxas keeps the branch, and skipped work costs no pipe time.  Taken
// branches cost a warp ~15-20 cycles each, so the unit of skipping is a whole block (2 x 3..4 fragments) on a cubelet,
// with three straight-line variants: both rows, only row 0, only row 1.
//
// gint_vlocal block, both rows: c[r][j] += a_r b_j over the two k-steps (x, y) of the cubelet.  All x-steps first: the two DMMAs
// of one accumulator are 2 N apart (a dependent DMMA waits 26 cycles, an independent one issues every 16).
template <int N>
__device__ __forceinline__ void vl_blk2(double (&c)[2][4][2], double a0x, double a0y, double a1x, double a1y, const double2 (&b)[4], int q) {
    if (N == 4) {
        asm volatile(
            "{\n\t.reg .pred pq;\n\tsetp.ne.s32 pq, %28, 0;\n\tL_%=:\n\t"
            GINT_DMMA("%0", "%1", "%16", "%20") GINT_DMMA("%8", "%9", "%18", "%20") GINT_DMMA("%2", "%3", "%16", "%22") GINT_DMMA("%10", "%11", "%18", "%22")
            GINT_DMMA("%4", "%5", "%16", "%24") GINT_DMMA("%12", "%13", "%18", "%24") GINT_DMMA("%6", "%7", "%16", "%26") GINT_DMMA("%14", "%15", "%18", "%26")
            GINT_DMMA("%0", "%1", "%17", "%21") GINT_DMMA("%8", "%9", "%19", "%21") GINT_DMMA("%2", "%3", "%17", "%23") GINT_DMMA("%10", "%11", "%19", "%23")
            GINT_DMMA("%4", "%5", "%17", "%25") GINT_DMMA("%12", "%13", "%19", "%25") GINT_DMMA("%6", "%7", "%17", "%27") GINT_DMMA("%14", "%15", "%19", "%27")
            "@pq bra.uni L_%=;\n\t}"
            : "+d"(c[0][0][0]), "+d"(c[0][0][1]), "+d"(c[0][1][0]), "+d"(c[0][1][1]), "+d"(c[0][2][0]), "+d"(c[0][2][1]), "+d"(c[0][3][0]), "+d"(c[0][3][1]),
              "+d"(c[1][0][0]), "+d"(c[1][0][1]), "+d"(c[1][1][0]), "+d"(c[1][1][1]), "+d"(c[1][2][0]), "+d"(c[1][2][1]), "+d"(c[1][3][0]), "+d"(c[1][3][1])
            : "d"(a0x), "d"(a0y), "d"(a1x), "d"(a1y), "d"(b[0].x), "d"(b[0].y), "d"(b[1].x), "d"(b[1].y), "d"(b[2].x), "d"(b[2].y), "d"(b[3].x), "d"(b[3].y), "r"(q));
    } else {
        asm volatile(
            "{\n\t.reg .pred pq;\n\tsetp.ne.s32 pq, %22, 0;\n\tL_%=:\n\t"
            GINT_DMMA("%0", "%1", "%12", "%16") GINT_DMMA("%6", "%7", "%14", "%16") GINT_DMMA("%2", "%3", "%12", "%18") GINT_DMMA("%8", "%9", "%14", "%18")
            GINT_DMMA("%4", "%5", "%12", "%20") GINT_DMMA("%10", "%11", "%14", "%20")
            GINT_DMMA("%0", "%1", "%13", "%17") GINT_DMMA("%6", "%7", "%15", "%17") GINT_DMMA("%2", "%3", "%13", "%19") GINT_DMMA("%8", "%9", "%15", "%19")
            GINT_DMMA("%4", "%5", "%13", "%21") GINT_DMMA("%10", "%11", "%15", "%21")
            "@pq bra.uni L_%=;\n\t}"
            : "+d"(c[0][0][0]), "+d"(c[0][0][1]), "+d"(c[0][1][0]), "+d"(c[0][1][1]), "+d"(c[0][2][0]), "+d"(c[0][2][1]),
              "+d"(c[1][0][0]), "+d"(c[1][0][1]), "+d"(c[1][1][0]), "+d"(c[1][1][1]), "+d"(c[1][2][0]), "+d"(c[1][2][1])
            : "d"(a0x), "d"(a0y), "d"(a1x), "d"(a1y), "d"(b[0].x), "d"(b[0].y), "d"(b[1].x), "d"(b[1].y), "d"(b[2].x), "d"(b[2].y), "r"(q));
    }
}
// one row of a block
template <int N>
__device__ __forceinline__ void vl_blk1(double (&c)[4][2], double ax, double ay, const double2 (&b)[4], int q) {
    if (N == 4) {
        asm volatile(
            "{\n\t.reg .pred pq;\n\tsetp.ne.s32 pq, %18, 0;\n\tL_%=:\n\t"
            GINT_DMMA("%0", "%1", "%8", "%10") GINT_DMMA("%2", "%3", "%8", "%12") GINT_DMMA("%4", "%5", "%8", "%14") GINT_DMMA("%6", "%7", "%8", "%16")
            GINT_DMMA("%0", "%1", "%9", "%11") GINT_DMMA("%2", "%3", "%9", "%13") GINT_DMMA("%4", "%5", "%9", "%15") GINT_DMMA("%6", "%7", "%9", "%17")
            "@pq bra.uni L_%=;\n\t}"
            : "+d"(c[0][0]), "+d"(c[0][1]), "+d"(c[1][0]), "+d"(c[1][1]), "+d"(c[2][0]), "+d"(c[2][1]), "+d"(c[3][0]), "+d"(c[3][1])
            : "d"(ax), "d"(ay), "d"(b[0].x), "d"(b[0].y), "d"(b[1].x), "d"(b[1].y), "d"(b[2].x), "d"(b[2].y), "d"(b[3].x), "d"(b[3].y), "r"(q));
    } else {
        asm volatile(
            "{\n\t.reg .pred pq;\n\tsetp.ne.s32 pq, %14, 0;\n\tL_%=:\n\t"
            GINT_DMMA("%0", "%1", "%6", "%8") GINT_DMMA("%2", "%3", "%6", "%10") GINT_DMMA("%4", "%5", "%6", "%12")
            GINT_DMMA("%0", "%1", "%7", "%9") GINT_DMMA("%2", "%3", "%7", "%11") GINT_DMMA("%4", "%5", "%7", "%13")
            "@pq bra.uni L_%=;\n\t}"
            : "+d"(c[0][0]), "+d"(c[0][1]), "+d"(c[1][0]), "+d"(c[1][1]), "+d"(c[2][0]), "+d"(c[2][1])
            : "d"(ax), "d"(ay), "d"(b[0].x), "d"(b[0].y), "d"(b[1].x), "d"(b[1].y), "d"(b[2].x), "d"(b[2].y), "r"(q));
    }
}
// Blocks of a consumer warp.
#define GINT_FRAG_BYTES (8 * GINT_ROW_BYTES)
struct Blk {
    unsigned oa, ob;                 // byte offsets of the first row fragment (side I) and of the first column fragment (side J) inside a cubelet of a stage
    unsigned d;                      // descriptor (PlanHdr::blk)
    __device__ __forceinline__ int row() const { return d & 15; }
    __device__ __forceinline__ bool has1() const { return (d >> 4) & 1u; }
    __device__ __forceinline__ int c0() const { return (d >> 5) & 15; }
    __device__ __forceinline__ int n() const { return (d >> 9) & 7; }
};
__device__ __forceinline__ Blk load_blk(const PlanHdr& X, unsigned desc) {
    Blk s; s.d = desc;
    s.oa = (unsigned)(s.row() * GINT_FRAG_BYTES);
    s.ob = (unsigned)((X.diag ? 0 : GINT_SLOT_MAX_BYTES) + s.c0() * GINT_FRAG_BYTES);
    return s;
}

// gint_vlocal, one block on one cubelet.  pa, pb: lane addresses of the first row fragment / first column fragment; ra, rb: the rows are active.
template <int NMAX>
__device__ __forceinline__ void vl_visit(double (&acc)[2][4][2], int n, unsigned pa, unsigned pb, int sx, int sy, bool ra, bool rb, int q) {
    double2 b[4];
#pragma unroll
    for (int j = 0; j < 4; j++) b[j] = make_double2(0.0, 0.0);
#pragma unroll
    for (int j = 0; j < NMAX; j++) b[j] = lds128(pb + j * GINT_FRAG_BYTES);
    double2 a0 = lds128(pa), a1 = lds128(pa + GINT_FRAG_BYTES);
    // sign of V at the lane's two points (sx, sy: 0 or 0x80000000): the orbital values carry sqrt(|V dV|)
    a0.x = __hiloint2double(__double2hiint(a0.x) ^ sx, __double2loint(a0.x)); a0.y = __hiloint2double(__double2hiint(a0.y) ^ sy, __double2loint(a0.y));
    a1.x = __hiloint2double(__double2hiint(a1.x) ^ sx, __double2loint(a1.x)); a1.y = __hiloint2double(__double2hiint(a1.y) ^ sy, __double2loint(a1.y));
    if (NMAX == 4 && n == 4) {
        if (ra && rb) vl_blk2<4>(acc, a0.x, a0.y, a1.x, a1.y, b, q);
        else if (ra) vl_blk1<4>(acc[0], a0.x, a0.y, b, q);
        else vl_blk1<4>(acc[1], a1.x, a1.y, b, q);
    } else {            // 3 columns (a narrower block of a small group runs its unused columns on whatever the slot holds there; never flushed)
        if (ra && rb) vl_blk2<3>(acc, a0.x, a0.y, a1.x, a1.y, b, q);
        else if (ra) vl_blk1<3>(acc[0], a0.x, a0.y, b, q);
        else vl_blk1<3>(acc[1], a1.x, a1.y, b, q);
    }
}
// gint_rho, one block on one ring stage (two cubelets): Y_qr = sum_j D[row r][column j] Phi_J[column j] at the 8 points of cubelet q
// (8 orbitals of I x 8 points), four accumulator chains (two with one row); the operands of Phi_J are loaded inside the block, so
// that ptxas schedules them among the DMMAs.  d[r][j][h]: stationary A operands (k-step h of column j); pj0, pj1: lane addresses of
// Phi_J[8 c0 + lane % 4][point lane / 4] in the two cubelets; y[q][r][e]: C fragments (orbital row lane / 4, points 2 (lane % 4) + e).
template <int R, int N>
__device__ __forceinline__ void rho_stage_blk(const double (&d)[2][4][2], unsigned pj0, unsigned pj1, int q, double (&y)[2][2][2]) {
    if (R == 2 && N == 4) {
        asm volatile(
            "{\n\t.reg .pred pq;\n\t.reg .f64 z;\n\t.reg .f64 b<16>;\n\tsetp.ne.s32 pq, %26, 0;\n\tmov.f64 z, 0d0000000000000000;\n\tL_%=:\n\t"
            "ld.shared.f64 b0, [%24+0];\n\tld.shared.f64 b1, [%24+256];\n\tld.shared.f64 b2, [%24+512];\n\tld.shared.f64 b3, [%24+768];\n\tld.shared.f64 b4, [%24+1024];\n\tld.shared.f64 b5, [%24+1280];\n\tld.shared.f64 b6, [%24+1536];\n\tld.shared.f64 b7, [%24+1792];\n\tld.shared.f64 b8, [%25+0];\n\tld.shared.f64 b9, [%25+256];\n\tld.shared.f64 b10, [%25+512];\n\tld.shared.f64 b11, [%25+768];\n\tld.shared.f64 b12, [%25+1024];\n\tld.shared.f64 b13, [%25+1280];\n\tld.shared.f64 b14, [%25+1536];\n\tld.shared.f64 b15, [%25+1792];\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%8},{b0},{z,z};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%16},{b0},{z,z};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%4,%5},{%8},{b8},{z,z};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%6,%7},{%16},{b8},{z,z};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%9},{b1},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%17},{b1},{%2,%3};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%4,%5},{%9},{b9},{%4,%5};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%6,%7},{%17},{b9},{%6,%7};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%10},{b2},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%18},{b2},{%2,%3};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%4,%5},{%10},{b10},{%4,%5};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%6,%7},{%18},{b10},{%6,%7};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%11},{b3},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%19},{b3},{%2,%3};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%4,%5},{%11},{b11},{%4,%5};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%6,%7},{%19},{b11},{%6,%7};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%12},{b4},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%20},{b4},{%2,%3};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%4,%5},{%12},{b12},{%4,%5};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%6,%7},{%20},{b12},{%6,%7};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%13},{b5},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%21},{b5},{%2,%3};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%4,%5},{%13},{b13},{%4,%5};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%6,%7},{%21},{b13},{%6,%7};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%14},{b6},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%22},{b6},{%2,%3};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%4,%5},{%14},{b14},{%4,%5};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%6,%7},{%22},{b14},{%6,%7};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%15},{b7},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%23},{b7},{%2,%3};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%4,%5},{%15},{b15},{%4,%5};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%6,%7},{%23},{b15},{%6,%7};\n\t"
            "@pq bra.uni L_%=;\n\t}"
            : "=d"(y[0][0][0]), "=d"(y[0][0][1]), "=d"(y[0][1][0]), "=d"(y[0][1][1]), "=d"(y[1][0][0]), "=d"(y[1][0][1]), "=d"(y[1][1][0]), "=d"(y[1][1][1])
            : "d"(d[0][0][0]), "d"(d[0][0][1]), "d"(d[0][1][0]), "d"(d[0][1][1]), "d"(d[0][2][0]), "d"(d[0][2][1]), "d"(d[0][3][0]), "d"(d[0][3][1]), "d"(d[1][0][0]), "d"(d[1][0][1]), "d"(d[1][1][0]), "d"(d[1][1][1]), "d"(d[1][2][0]), "d"(d[1][2][1]), "d"(d[1][3][0]), "d"(d[1][3][1]), "r"(pj0), "r"(pj1), "r"(q));
    } else if (R == 2) {
        asm volatile(
            "{\n\t.reg .pred pq;\n\t.reg .f64 z;\n\t.reg .f64 b<12>;\n\tsetp.ne.s32 pq, %22, 0;\n\tmov.f64 z, 0d0000000000000000;\n\tL_%=:\n\t"
            "ld.shared.f64 b0, [%20+0];\n\tld.shared.f64 b1, [%20+256];\n\tld.shared.f64 b2, [%20+512];\n\tld.shared.f64 b3, [%20+768];\n\tld.shared.f64 b4, [%20+1024];\n\tld.shared.f64 b5, [%20+1280];\n\tld.shared.f64 b6, [%21+0];\n\tld.shared.f64 b7, [%21+256];\n\tld.shared.f64 b8, [%21+512];\n\tld.shared.f64 b9, [%21+768];\n\tld.shared.f64 b10, [%21+1024];\n\tld.shared.f64 b11, [%21+1280];\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%8},{b0},{z,z};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%14},{b0},{z,z};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%4,%5},{%8},{b6},{z,z};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%6,%7},{%14},{b6},{z,z};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%9},{b1},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%15},{b1},{%2,%3};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%4,%5},{%9},{b7},{%4,%5};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%6,%7},{%15},{b7},{%6,%7};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%10},{b2},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%16},{b2},{%2,%3};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%4,%5},{%10},{b8},{%4,%5};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%6,%7},{%16},{b8},{%6,%7};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%11},{b3},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%17},{b3},{%2,%3};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%4,%5},{%11},{b9},{%4,%5};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%6,%7},{%17},{b9},{%6,%7};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%12},{b4},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%18},{b4},{%2,%3};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%4,%5},{%12},{b10},{%4,%5};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%6,%7},{%18},{b10},{%6,%7};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%13},{b5},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%19},{b5},{%2,%3};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%4,%5},{%13},{b11},{%4,%5};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%6,%7},{%19},{b11},{%6,%7};\n\t"
            "@pq bra.uni L_%=;\n\t}"
            : "=d"(y[0][0][0]), "=d"(y[0][0][1]), "=d"(y[0][1][0]), "=d"(y[0][1][1]), "=d"(y[1][0][0]), "=d"(y[1][0][1]), "=d"(y[1][1][0]), "=d"(y[1][1][1])
            : "d"(d[0][0][0]), "d"(d[0][0][1]), "d"(d[0][1][0]), "d"(d[0][1][1]), "d"(d[0][2][0]), "d"(d[0][2][1]), "d"(d[1][0][0]), "d"(d[1][0][1]), "d"(d[1][1][0]), "d"(d[1][1][1]), "d"(d[1][2][0]), "d"(d[1][2][1]), "r"(pj0), "r"(pj1), "r"(q));
    } else if (N == 4) {
        asm volatile(
            "{\n\t.reg .pred pq;\n\t.reg .f64 z;\n\t.reg .f64 b<16>;\n\tsetp.ne.s32 pq, %14, 0;\n\tmov.f64 z, 0d0000000000000000;\n\tL_%=:\n\t"
            "ld.shared.f64 b0, [%12+0];\n\tld.shared.f64 b1, [%12+256];\n\tld.shared.f64 b2, [%12+512];\n\tld.shared.f64 b3, [%12+768];\n\tld.shared.f64 b4, [%12+1024];\n\tld.shared.f64 b5, [%12+1280];\n\tld.shared.f64 b6, [%12+1536];\n\tld.shared.f64 b7, [%12+1792];\n\tld.shared.f64 b8, [%13+0];\n\tld.shared.f64 b9, [%13+256];\n\tld.shared.f64 b10, [%13+512];\n\tld.shared.f64 b11, [%13+768];\n\tld.shared.f64 b12, [%13+1024];\n\tld.shared.f64 b13, [%13+1280];\n\tld.shared.f64 b14, [%13+1536];\n\tld.shared.f64 b15, [%13+1792];\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%4},{b0},{z,z};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%4},{b8},{z,z};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%5},{b1},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%5},{b9},{%2,%3};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%6},{b2},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%6},{b10},{%2,%3};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%7},{b3},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%7},{b11},{%2,%3};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%8},{b4},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%8},{b12},{%2,%3};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%9},{b5},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%9},{b13},{%2,%3};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%10},{b6},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%10},{b14},{%2,%3};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%11},{b7},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%11},{b15},{%2,%3};\n\t"
            "@pq bra.uni L_%=;\n\t}"
            : "=d"(y[0][0][0]), "=d"(y[0][0][1]), "=d"(y[1][0][0]), "=d"(y[1][0][1])
            : "d"(d[0][0][0]), "d"(d[0][0][1]), "d"(d[0][1][0]), "d"(d[0][1][1]), "d"(d[0][2][0]), "d"(d[0][2][1]), "d"(d[0][3][0]), "d"(d[0][3][1]), "r"(pj0), "r"(pj1), "r"(q));
    } else {
        asm volatile(
            "{\n\t.reg .pred pq;\n\t.reg .f64 z;\n\t.reg .f64 b<12>;\n\tsetp.ne.s32 pq, %12, 0;\n\tmov.f64 z, 0d0000000000000000;\n\tL_%=:\n\t"
            "ld.shared.f64 b0, [%10+0];\n\tld.shared.f64 b1, [%10+256];\n\tld.shared.f64 b2, [%10+512];\n\tld.shared.f64 b3, [%10+768];\n\tld.shared.f64 b4, [%10+1024];\n\tld.shared.f64 b5, [%10+1280];\n\tld.shared.f64 b6, [%11+0];\n\tld.shared.f64 b7, [%11+256];\n\tld.shared.f64 b8, [%11+512];\n\tld.shared.f64 b9, [%11+768];\n\tld.shared.f64 b10, [%11+1024];\n\tld.shared.f64 b11, [%11+1280];\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%4},{b0},{z,z};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%4},{b6},{z,z};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%5},{b1},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%5},{b7},{%2,%3};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%6},{b2},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%6},{b8},{%2,%3};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%7},{b3},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%7},{b9},{%2,%3};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%8},{b4},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%8},{b10},{%2,%3};\n\t"
            "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%9},{b5},{%0,%1};\n\tmma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%2,%3},{%9},{b11},{%2,%3};\n\t"
            "@pq bra.uni L_%=;\n\t}"
            : "=d"(y[0][0][0]), "=d"(y[0][0][1]), "=d"(y[1][0][0]), "=d"(y[1][0][1])
            : "d"(d[0][0][0]), "d"(d[0][0][1]), "d"(d[0][1][0]), "d"(d[0][1][1]), "d"(d[0][2][0]), "d"(d[0][2][1]), "r"(pj0), "r"(pj1), "r"(q));
    }
}
// One block on one stage, then rho_g += sum_i Phi_I[i][g] Y[i][g] (the sum over the 8 orbital rows of a fragment = over lane / 4 is
// taken once per stage by the caller).  pi: lane address of Phi_I[8 row + lane / 4][points 2 (lane % 4), + 1] in cubelet 0.
// Columns beyond the block's n hold D = 0 and whatever the ring holds there (always finite: the ring starts zeroed and only ever
// receives orbital values), likewise the second row of a single-row block.
template <int NMAX>
__device__ __forceinline__ void rho_stage_issue(const double (&d)[2][4][2], int n, bool has1, unsigned pj, int q, double (&y)[2][2][2]) {
    const bool wide = NMAX == 4 && n == 4;
    const unsigned pj1 = pj + 2 * GINT_SLOT_MAX_BYTES;
    if (has1) {
        if (wide) rho_stage_blk<2, 4>(d, pj, pj1, q, y); else rho_stage_blk<2, 3>(d, pj, pj1, q, y);
    } else {
        y[0][1][0] = 0.0; y[0][1][1] = 0.0; y[1][1][0] = 0.0; y[1][1][1] = 0.0;
        if (wide) rho_stage_blk<1, 4>(d, pj, pj1, q, y); else rho_stage_blk<1, 3>(d, pj, pj1, q, y);
    }
}
__device__ __forceinline__ void rho_stage_retire(const double (&y)[2][2][2], unsigned pi, double (&part)[GINT_SC][2]) {
    const unsigned pi1 = pi + 2 * GINT_SLOT_MAX_BYTES;
    const double2 f00 = lds128(pi), f01 = lds128(pi + GINT_FRAG_BYTES), f10 = lds128(pi1), f11 = lds128(pi1 + GINT_FRAG_BYTES);
    part[0][0] = fma(y[0][0][0], f00.x, part[0][0]); part[0][1] = fma(y[0][0][1], f00.y, part[0][1]);
    part[1][0] = fma(y[1][0][0], f10.x, part[1][0]); part[1][1] = fma(y[1][0][1], f10.y, part[1][1]);
    part[0][0] = fma(y[0][1][0], f01.x, part[0][0]); part[0][1] = fma(y[0][1][1], f01.y, part[0][1]);
    part[1][0] = fma(y[1][1][0], f11.x, part[1][0]); part[1][1] = fma(y[1][1][1], f11.y, part[1][1]);
}
// stationary operands of a row fragment (gint_rho): d[j][h] = Dh[orbital row 8 row + lr of I][orbital column 8 (c0 + j) + 4 h + lc of J]
__device__ __forceinline__ void load_drow(const PlanHdr& X, int rowf, int c0, int n, const double* __restrict__ Dh, double (&d)[4][2]) {
    const int lane = threadIdx.x & 31, lr = lane >> 2, lc = lane & 3;
    const int row = 8 * rowf + lr;
    const int a = row < GINT_TILE_ORB ? X.row_atom[0][row] : 255, oa = row < GINT_TILE_ORB ? X.row_orb[0][row] : 0;
#pragma unroll
    for (int j = 0; j < 4; j++)
#pragma unroll
        for (int h = 0; h < 2; h++) {
            double v = 0.0;
            if (j < n && a != 255) {
                const int col = 8 * (c0 + j) + 4 * h + lc;
                const int bb = X.row_atom[1][col];
                if (bb != 255) {
                    const PairEnt pe = X.pair[a][bb];
                    if (pe.off != 0xffffffffu) v = __ldg(Dh + pe.off + oa * pe.sr + X.row_orb[1][col] * pe.sc);
                }
            }
            d[j][h] = v;
        }
}
// flush of a row fragment's accumulators (gint_vlocal): element (row, col) -> atom pair (a, b), orbitals (oa, ob) -> canonical block
// (transposed if the canonical key is (b, a)).  Exact zeros (fragments never touched, atoms that do not overlap inside this batch) are skipped.
__device__ __forceinline__ void flush_row(const PlanHdr& X, int rowf, int c0, int n, const double (&acc)[4][2], double* __restrict__ Hc) {
    const int lane = threadIdx.x & 31, lr = lane >> 2, lc = lane & 3;
    const int row = 8 * rowf + lr;
    const int a = X.row_atom[0][row], oa = X.row_orb[0][row];
    if (a == 255) return;
#pragma unroll
    for (int j = 0; j < 4; j++) {
        if (j >= n) break;
#pragma unroll
        for (int e = 0; e < 2; e++) {
            const double v = acc[j][e];
            const int col = 8 * (c0 + j) + 2 * lc + e;
            const int bb = X.row_atom[1][col], ob = X.row_orb[1][col];
            if (bb == 255 || v == 0.0) continue;
            const PairEnt pe = X.pair[a][bb];
            if (pe.off == 0xffffffffu) continue;
            atomicAdd(Hc + pe.off + oa * pe.sr + ob * pe.sc, v);
        }
    }
}

template <bool VLOCAL>
__device__ __forceinline__ void consumer_role(TileSmem& S, const double* __restrict__ Dh, double* __restrict__ Hc) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, lr = lane >> 2, lc = lane & 3;
    const unsigned ring0 = smem_addr(&S.ring[0][0]);
    // lane parts of the operand addresses
    // (gint_rho: with the swizzle of the slot rows, see k_eval_phi; fragments start at multiples of 8 rows)
    const unsigned lane_v = lr * GINT_ROW_BYTES + ((VLOCAL ? lc : (lc ^ (lr & 2))) * 16);  // row lr of a fragment, points 2 lc, 2 lc + 1
    const unsigned lane_j = lc * GINT_ROW_BYTES + ((lr ^ ((lc & 2) << 1)) * 8);            // gint_rho B operand: row lc of the k-step, point lr
    // ring position of the next stage: slot, parity of its full barrier, and the slot's addresses (all 32-bit shared addresses)
    constexpr unsigned NSK = VLOCAL ? GINT_NS : GINT_NS - GINT_RHO_RSV;
    unsigned rs = 0, rph = 0;
    int gsl = 0;                                                           // gint_rho: stages done (selects the lane-partial buffer)
    const unsigned full0 = smem_addr(&S.full[0]), empty0 = smem_addr(&S.empty[0]);
    // gint_rho: where the lane's reduced partial density of a stage goes (see the butterfly below)
    const unsigned lpart0 = smem_addr(&S.ring[GINT_NS - GINT_RHO_RSV][0]) + (unsigned)(warp * 32 + lane) * (GINT_SC * 2 * 8);
    const unsigned lfull0 = smem_addr(&S.lfull[0]), lempty0 = smem_addr(&S.lempty[0]);
#ifdef GINT_DBG_STATS
    unsigned long long dbg_acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
#endif
    for (int t = 0;; t++) {
        const int c = t % GINT_NCTX;
        DBG_T(t_ctx0);
        mbar_wait(&S.ctx_full[c], (t / GINT_NCTX) & 1);
        const PlanHdr& X = plan_hdr(S, c);
        if (!X.valid) break;
        DBG_T(t_tile0);
        DBG_ADD(7, t_tile0 - t_ctx0);
        Blk bk[GINT_WARP_BLOCKS];
        double acc[GINT_WARP_BLOCKS][2][4][2];      // gint_vlocal: accumulators; gint_rho: stationary D operands (column 3 of blocks 1, 2 is never touched)
        const int q = X.zero;
#pragma unroll
        for (int k = 0; k < GINT_WARP_BLOCKS; k++) {
            bk[k] = load_blk(X, X.blk[k][warp]);
            if (VLOCAL) {
#pragma unroll
                for (int j = 0; j < 4; j++) { acc[k][0][j][0] = 0.0; acc[k][0][j][1] = 0.0; acc[k][1][j][0] = 0.0; acc[k][1][j][1] = 0.0; }
            } else {
                load_drow(X, bk[k].row(), bk[k].c0(), bk[k].n(), Dh, acc[k][0]);
                load_drow(X, bk[k].row() + 1, bk[k].c0(), bk[k].has1() ? bk[k].n() : 0, Dh, acc[k][1]);
            }
        }
        const int nstage = X.nstage;
        const unsigned vis0 = smem_addr(&plan_cub(S, c)[0].vis[warp]);
        const unsigned sgn_off = (unsigned)X.RI * GINT_ROW_BYTES + lc * 16;    // gint_vlocal: the lane's two points in the sign row of slot I
        unsigned cur[GINT_SC], nxt[GINT_SC];
#pragma unroll
        for (int qq = 0; qq < GINT_SC; qq++) cur[qq] = lds_u8(vis0 + qq * (unsigned)sizeof(PlanCub));
        DBG_T(t_tile1);
        DBG_ADD(0, t_tile1 - t_tile0);
        unsigned visp = vis0 + GINT_SC * (unsigned)sizeof(PlanCub);           // visit codes of the next stage
        for (int st = 0; st < nstage; st++) {
            const unsigned s = rs;
            DBG_T(t_w0);
            mbar_wait_s(full0 + 8 * s, rph);
            DBG_T(t_w1);
            DBG_ADD(1, t_w1 - t_w0);
            double part[GINT_SC][2];
#pragma unroll
            for (int qq = 0; qq < GINT_SC; qq++) { part[qq][0] = 0.0; part[qq][1] = 0.0; nxt[qq] = lds_u8(visp + qq * (unsigned)sizeof(PlanCub)); }
            visp += GINT_SC * (unsigned)sizeof(PlanCub);
#ifdef GINT_DBG_WARPS
            if (warp < GINT_DBG_WARPS)        // developer switch: only the first warps work (serial time of a warp without competition for the pipe)
#endif
#ifndef GINT_DBG_NO_MMA
            if (VLOCAL) {
#pragma unroll
                for (int qq = 0; qq < GINT_SC; qq++) {
                    const unsigned code = cur[qq];
                    if (code) {
                        const unsigned base = ring0 + s * GINT_STAGE_BYTES + qq * 2 * GINT_SLOT_MAX_BYTES;
                        const double2 sg = lds128(base + sgn_off);
                        const int sx = __double2hiint(sg.x), sy = __double2hiint(sg.y);
#pragma unroll
                        for (int k = 0; k < GINT_WARP_BLOCKS; k++) {
                            const unsigned rr = (code >> (2 * k)) & 3u;
                            if (rr) {
                                DBG_ADD(6, (rr == 3u ? 4 : 2) * bk[k].n());
                                if (k == 0) vl_visit<4>(acc[k], bk[k].n(), base + bk[k].oa + lane_v, base + bk[k].ob + lane_v, sx, sy, rr & 1u, rr & 2u, q);
                                else vl_visit<3>(acc[k], bk[k].n(), base + bk[k].oa + lane_v, base + bk[k].ob + lane_v, sx, sy, rr & 1u, rr & 2u, q);
                            }
                        }
                    }
                }
            } else {
                // a block is worked on the whole stage if one of its rows and one of its columns are active on one of the two cubelets
                const unsigned code = cur[0] | cur[GINT_SC - 1];
                const unsigned base = ring0 + s * GINT_STAGE_BYTES;
                double y[2][2][2];
                unsigned pend = 0;              // lane address of the Phi_I rows of the block whose Y is still to be used (0: none)
#pragma unroll
                for (int k = 0; k < GINT_WARP_BLOCKS; k++) {
                    if ((code >> (2 * k)) & 3u) {
                        DBG_ADD(6, (bk[k].has1() ? 8 : 4) * bk[k].n());
                        if (pend) rho_stage_retire(y, pend, part);
                        if (k == 0) rho_stage_issue<4>(acc[k], bk[k].n(), bk[k].has1(), base + bk[k].ob + lane_j, q, y);
                        else rho_stage_issue<3>(acc[k], bk[k].n(), bk[k].has1(), base + bk[k].ob + lane_j, q, y);
                        pend = base + bk[k].oa + lane_v;
                    }
                }
                if (pend) rho_stage_retire(y, pend, part);
            }
#endif
            if (!VLOCAL) {
                // part[q][e]: point 2 lc + e of cubelet q, partial over the lane's orbital row: handed to a reducer warp as it is
                const unsigned lb = (unsigned)gsl % GINT_NBUF;
                DBG_T(t_l0);
                if (gsl >= GINT_NBUF) mbar_wait_s(lempty0 + 8 * lb, (unsigned)((gsl / GINT_NBUF) - 1) & 1u);
                DBG_T(t_l1);
                DBG_ADD(3, t_l1 - t_l0);
                const unsigned dst = lpart0 + lb * GINT_LPART_BYTES;
                asm volatile("st.shared.v2.f64 [%0], {%1, %2};" :: "r"(dst), "d"(part[0][0]), "d"(part[0][1]) : "memory");
                asm volatile("st.shared.v2.f64 [%0], {%1, %2};" :: "r"(dst + 16), "d"(part[GINT_SC - 1][0]), "d"(part[GINT_SC - 1][1]) : "memory");
                __syncwarp();
                if (lane == 0) mbar_arrive_s(lfull0 + 8 * lb);
                gsl++;
            }
            __syncwarp();
            if (lane == 0) mbar_arrive_s(empty0 + 8 * s);
            if (++rs == NSK) { rs = 0; rph ^= 1u; }
#pragma unroll
            for (int qq = 0; qq < GINT_SC; qq++) cur[qq] = nxt[qq];
            DBG_T(t_w2);
            DBG_ADD(2, t_w2 - t_w1);
        }
        DBG_T(t_loop);
        if (VLOCAL) {
#pragma unroll
            for (int k = 0; k < GINT_WARP_BLOCKS; k++) {
                if (bk[k].n() == 0) continue;
                flush_row(X, bk[k].row(), bk[k].c0(), bk[k].n(), acc[k][0], Hc);
                if (bk[k].has1()) flush_row(X, bk[k].row() + 1, bk[k].c0(), bk[k].n(), acc[k][1], Hc);
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&S.ctx_free[c]);
        DBG_T(t_end);
        DBG_ADD(3, t_end - t_loop);
        DBG_ADD(4, t_end - t_tile0);
        DBG_ADD(5, 1);
    }
#ifdef GINT_DBG_STATS
    if (lane == 0) for (int i = 0; i < 8; i++) { atomicAdd(&g_dbg[i], dbg_acc[i]); atomicAdd(&g_dbgw[warp][i], dbg_acc[i]); }
#endif
}

// ---------------------------------------------------------------------------------------------------
// gint_vlocal / gint_rho main kernels (north_star step 3): persistent, one CTA per SM.
template <bool VLOCAL>
__global__ void __launch_bounds__(GINT_CTA_THREADS, 1)
k_tiles(Geom g, const unsigned char* __restrict__ plan, const unsigned* __restrict__ planoff /* of the wave's first tile */, int n_tiles,
        int* __restrict__ queue, u64 wave_row0, const double* __restrict__ phi, const double* __restrict__ Dh, double* __restrict__ out /* Hc or rho */) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    TileSmem& S = *reinterpret_cast<TileSmem*>((reinterpret_cast<uintptr_t>(smem_raw) + 127) & ~(uintptr_t)127);
    const int warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
        for (int s = 0; s < GINT_NS; s++) { mbar_init(&S.full[s], 1); mbar_init(&S.empty[s], GINT_MMA_WARPS); }
        for (int c = 0; c < GINT_NCTX; c++) { mbar_init(&S.ctx_full[c], 1); mbar_init(&S.ctx_free[c], GINT_MMA_WARPS + 1 + (VLOCAL ? 0 : GINT_NRED)); }
        for (int k = 0; k < GINT_NBUF; k++) { mbar_init(&S.lfull[k], GINT_MMA_WARPS); mbar_init(&S.lempty[k], 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // the ring starts zeroed: the consumers may read rows of a stage that no copy has written yet (multiplied by zeros: must be finite)
    for (unsigned i = threadIdx.x; i < sizeof(S.ring) / 16; i += GINT_CTA_THREADS) reinterpret_cast<uint4*>(&S.ring[0][0])[i] = make_uint4(0u, 0u, 0u, 0u);
    // generic-proxy stores above, async-proxy (cp.async.bulk) writes to the same bytes later: order the two proxies
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
    if (warp < GINT_MMA_WARPS) {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" :: "n"(GINT_REGS_MMA));
        consumer_role<VLOCAL>(S, Dh, out);
    } else {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" :: "n"(GINT_REGS_AUX));
        if (warp == GINT_MMA_WARPS) issuer_role<VLOCAL>(g, S, plan, planoff, n_tiles, queue, phi, wave_row0, out);
        else if (!VLOCAL && warp - GINT_MMA_WARPS - 1 < GINT_NRED) reducer_role(g, S, warp - GINT_MMA_WARPS - 1, out);
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
// Phi layout (gint_init): rows of every (batch, group) slot array = (cubelets on which the group is active) x (orbital rows
// padded to whole fragments + the sign row).  One thread per batch.
__global__ void __launch_bounds__(128) k_phi_rows(long long n_batch_total, const int* __restrict__ bstart, const NeighEntry* __restrict__ bent,
                                                  const int* __restrict__ gstart, const int* __restrict__ atom_spec,
                                                  const SpeciesDev* __restrict__ sp, unsigned* __restrict__ grows) {
    const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= n_batch_total) return;
    const int e0 = bstart[b], n = bstart[b + 1] - e0, G = gstart[b + 1] - gstart[b];
    for (int k = 0; k < G; k++) {
        cmask m = czero();
        int rows = 0;
        for (int e = group_begin(k, n, G); e < group_begin(k + 1, n, G); e++) {
            const NeighEntry en = bent[e0 + e];
            m |= cmask{en.mask[0], en.mask[1]};
            rows += sp[atom_spec[en.atom]].norb;
        }
        grows[gstart[b] + k] = (unsigned)(ccount(m) * (((rows + 7) & ~7) + 1));       // + the sign row
    }
}

int gint_build_phi_layout(gint_ctx* c, const int* d_bgroups, size_t phi_cap_bytes, bool* batch_too_big) {
    (void)d_bgroups;
    *batch_too_big = false;
    const long long nbt = c->n_batch_total;
    std::vector<int> gs(nbt + 1);
    GINT_CUDA(cudaMemcpy(gs.data(), c->d_gstart, sizeof(int) * (nbt + 1), cudaMemcpyDeviceToHost));
    const long long ng = gs[nbt];
    unsigned* d_grows = nullptr;
    GINT_CUDA(cudaMalloc(&d_grows, sizeof(unsigned) * (ng ? ng : 1)));
    if (nbt > 0) k_phi_rows<<<(unsigned)((nbt + 127) / 128), 128>>>(nbt, c->d_bstart, c->d_bent, c->d_gstart, c->d_atom_species, c->d_species, d_grows);
    GINT_CUDA(cudaGetLastError());
    std::vector<unsigned> grows(ng);
    if (ng) GINT_CUDA(cudaMemcpy(grows.data(), d_grows, sizeof(unsigned) * ng, cudaMemcpyDeviceToHost));
    GINT_CUDA(cudaFree(d_grows));
    std::vector<unsigned long long> goff(ng + 1);
    unsigned long long acc = 0;
    for (long long i = 0; i < ng; i++) { goff[i] = acc; acc += grows[i]; }
    goff[ng] = acc;
    c->phi_rows_total = acc;
    std::vector<int> ts(nbt + 1);
    GINT_CUDA(cudaMemcpy(ts.data(), c->d_tstart, sizeof(int) * (nbt + 1), cudaMemcpyDeviceToHost));
    // waves: contiguous batch ranges of at most cap rows
    const unsigned long long cap_rows = std::max<unsigned long long>(phi_cap_bytes / GINT_ROW_BYTES, 1);
    c->waves.clear();
    unsigned long long max_rows = 0;
    long long b = 0;
    while (b < nbt) {
        gint_ctx::Wave w; w.b0 = b; w.row0 = goff[gs[b]];
        unsigned long long rows = 0;
        while (b < nbt) {
            const unsigned long long br = goff[gs[b + 1]] - goff[gs[b]];
            if (br > cap_rows) { *batch_too_big = true; GINT_FAIL(GINT_ERR_OUT_OF_MEMORY, "orbital values of one batch (%llu bytes) exceed the scratch buffer (%zu bytes)", br * GINT_ROW_BYTES, phi_cap_bytes); }
            if (rows + br > cap_rows) break;
            rows += br; b++;
        }
        w.b1 = b; w.rows = rows; w.t0 = ts[w.b0]; w.t1 = ts[w.b1];
        if (w.t1 > w.t0) { c->waves.push_back(w); max_rows = std::max(max_rows, rows); }
    }
    goff.pop_back();
    if (goff.empty()) goff.push_back(0);
    GINT_CUDA(cudaMalloc((void**)&c->d_goff, sizeof(unsigned long long) * goff.size()));
    GINT_CUDA(cudaMemcpy(c->d_goff, goff.data(), sizeof(unsigned long long) * goff.size(), cudaMemcpyHostToDevice));
    c->device_bytes += sizeof(unsigned long long) * goff.size();
    c->phi_bytes = (size_t)std::max<unsigned long long>(max_rows, 1) * GINT_ROW_BYTES;
    GINT_CUDA(cudaMalloc((void**)&c->d_phi, c->phi_bytes));
    c->device_bytes += c->phi_bytes;
    GINT_CUDA(cudaMalloc((void**)&c->d_queue, sizeof(int) * (c->waves.size() + 1)));
    if (!c->copy_stream) GINT_CUDA(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
    for (auto& e : c->ev_copy) if (e) cudaEventDestroy(e);
    c->ev_copy.assign(c->waves.size() + 1, nullptr);
    for (auto& e : c->ev_copy) GINT_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    for (int k = 0; k < 2; k++) {
        c->ev_wave[k].assign(2 * c->waves.size(), nullptr);
        for (auto& e : c->ev_wave[k]) GINT_CUDA(cudaEventCreate(&e));
    }
    return GINT_OK;
}

// Tile plans: sizes, offsets, contents.  The tile list itself is not needed afterwards.
int gint_build_plans(gint_ctx* c) {
    const long long nt = c->n_tiles;
    int* d_units = nullptr;
    GINT_CUDA(cudaMalloc(&d_units, sizeof(int) * (size_t)(nt ? nt : 1)));
    GINT_CUDA(cudaMalloc((void**)&c->d_planoff, sizeof(unsigned) * (size_t)(nt + 1)));
    c->device_bytes += sizeof(unsigned) * (size_t)(nt + 1);
    if (nt > 0) k_plan_count<<<(unsigned)((nt + 255) / 256), 256>>>(nt, c->d_tile, c->d_bstart, c->d_bent, d_units);
    GINT_CUDA(cudaGetLastError());
    long long total = 0;
    int rc = gint_device_excl_scan(d_units, nt, reinterpret_cast<int*>(c->d_planoff), &total);
    cudaFree(d_units);
    if (rc) return rc;
    c->plan_bytes = (size_t)total * 16;
    GINT_CUDA(cudaMalloc((void**)&c->d_plan, c->plan_bytes ? c->plan_bytes : 16));
    c->device_bytes += c->plan_bytes;
    if (nt > 0)
        k_plan_fill<<<(unsigned)nt, GINT_PLAN_THREADS>>>(c->geom, c->d_tile, c->d_bstart, c->d_bent, c->d_gstart, c->d_goff, c->d_atom_species,
                                                          c->d_species, c->d_crow, c->d_ckey, c->d_coff, c->d_planoff, c->d_plan);
    GINT_CUDA(cudaGetLastError());
    GINT_CUDA(cudaDeviceSynchronize());
    cudaFree(c->d_tile); c->d_tile = nullptr;
    c->device_bytes -= sizeof(int2) * (size_t)(nt ? nt : 1);
    return GINT_OK;
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
                double ax, ay, az;
                image_pos(g, atom_pos + 3 * en.atom, t1, t2, t3, ax, ay, az);
                const double dx = x - ax, dy = y - ay, dz = z - az;
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
    // per function and device, not per context: set to what the kernels can ever need on this device
    cudaDeviceProp prop;
    GINT_CUDA(cudaGetDeviceProperties(&prop, c->device));
    const int lim = (int)prop.sharedMemPerBlockOptin;
    GINT_CUDA(cudaFuncSetAttribute(k_tiles<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim));
    GINT_CUDA(cudaFuncSetAttribute(k_tiles<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim));
    GINT_CUDA(cudaFuncSetAttribute(k_eval_phi<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim));
    GINT_CUDA(cudaFuncSetAttribute(k_eval_phi<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim));
    GINT_CUDA(cudaFuncSetAttribute(k_eval_phi<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim));
    GINT_CUDA(cudaFuncSetAttribute(k_eval_phi<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim));
    c->n_sm = prop.multiProcessorCount;
    return GINT_OK;
}

// Mesh planes (index along a1) below which every point belongs to a batch before batch b (batches are numbered a1-major).
static long long planes_before(const gint_ctx* c, long long b) {
    const Geom& g = c->geom;
    const long long per_plane = (long long)g.nb[1] * g.nb[2];
    return std::min<long long>((b / per_plane) * g.bs[0], g.N[0]);
}
// ... and the planes that hold the points of all batches before b (the plane of batch b - 1 included)
static long long planes_through(const gint_ctx* c, long long b) {
    const Geom& g = c->geom;
    const long long per_plane = (long long)g.nb[1] * g.nb[2];
    return b <= 0 ? 0 : std::min<long long>(((b - 1) / per_plane + 1) * g.bs[0], g.N[0]);
}

// one wave: evaluate the orbital values of its batches, then contract its tiles.
// Host path (h_in / h_out != nullptr): gint_vlocal copies the planes of V a wave needs on the copy stream, all waves ahead of the
// kernels; gint_rho copies the planes of rho a wave has completed back while the next wave runs.
template <bool VLOCAL>
static int launch_waves(gint_ctx* c, const double* in, double* out, cudaStream_t st, const double* h_in, double* h_out) {
    if (c->waves.empty()) return GINT_OK;
    GINT_CUDA(cudaMemsetAsync(c->d_queue, 0, sizeof(int) * c->waves.size(), st));
    const int tab_cells = (int)(c->tab_bytes / 16);
    const size_t plane = (size_t)c->geom.N[1] * c->geom.N[2];
    const size_t nw = c->waves.size();
    cudaStream_t cs = c->copy_stream;
    if (VLOCAL && h_in) {
        // the copy stream starts where the caller's stream stands, then runs ahead
        GINT_CUDA(cudaEventRecord(c->ev_copy[nw], st));
        GINT_CUDA(cudaStreamWaitEvent(cs, c->ev_copy[nw], 0));
        long long done = 0;
        for (size_t w = 0; w < nw; w++) {
            const long long upto = w + 1 == nw ? c->geom.N[0] : planes_through(c, c->waves[w].b1);
            if (upto > done) GINT_CUDA(cudaMemcpyAsync(const_cast<double*>(in) + done * plane, h_in + done * plane, sizeof(double) * (upto - done) * plane, cudaMemcpyHostToDevice, cs));
            done = std::max(done, upto);
            GINT_CUDA(cudaEventRecord(c->ev_copy[w], cs));
        }
    }
    long long copied = 0;
    for (size_t w = 0; w < nw; w++) {
        const gint_ctx::Wave& W = c->waves[w];
        const unsigned nb = (unsigned)(W.b1 - W.b0);
        if (VLOCAL && h_in) GINT_CUDA(cudaStreamWaitEvent(st, c->ev_copy[w], 0));
        if (c->tab_in_smem)
            k_eval_phi<true, VLOCAL><<<nb, GINT_EVAL_THREADS, c->smem_eval, st>>>(c->geom, W.b0, c->d_bstart, c->d_bent, c->d_gstart, c->d_goff, W.row0,
                c->d_atom_pos, c->d_atom_species, c->d_species, c->d_tab, tab_cells, VLOCAL ? in : nullptr, c->d_phi);
        else
            k_eval_phi<false, VLOCAL><<<nb, GINT_EVAL_THREADS, c->smem_eval, st>>>(c->geom, W.b0, c->d_bstart, c->d_bent, c->d_gstart, c->d_goff, W.row0,
                c->d_atom_pos, c->d_atom_species, c->d_species, c->d_tab, tab_cells, VLOCAL ? in : nullptr, c->d_phi);
        GINT_CUDA(cudaGetLastError());
        GINT_CUDA(cudaEventRecord(c->ev_wave[VLOCAL ? 0 : 1][2 * w], st));
        const int nt = (int)(W.t1 - W.t0);
        const unsigned grid = (unsigned)std::min<long long>(c->n_sm, nt);
        k_tiles<VLOCAL><<<grid, GINT_CTA_THREADS, c->smem_bytes, st>>>(c->geom, c->d_plan, c->d_planoff + W.t0, nt, c->d_queue + w, W.row0, c->d_phi,
                                                                       VLOCAL ? nullptr : in, out);
        GINT_CUDA(cudaGetLastError());
        GINT_CUDA(cudaEventRecord(c->ev_wave[VLOCAL ? 0 : 1][2 * w + 1], st));
        if (!VLOCAL && h_out) {
            // the planes no later wave adds to
            const long long upto = w + 1 == nw ? c->geom.N[0] : planes_before(c, c->waves[w + 1].b0);
            GINT_CUDA(cudaEventRecord(c->ev_copy[w], st));
            GINT_CUDA(cudaStreamWaitEvent(cs, c->ev_copy[w], 0));
            if (upto > copied) GINT_CUDA(cudaMemcpyAsync(h_out + copied * plane, out + copied * plane, sizeof(double) * (upto - copied) * plane, cudaMemcpyDeviceToHost, cs));
            copied = std::max(copied, upto);
        }
    }
    if (!VLOCAL && h_out) {         // the caller's stream ends behind the last copy
        GINT_CUDA(cudaEventRecord(c->ev_copy[nw], cs));
        GINT_CUDA(cudaStreamWaitEvent(st, c->ev_copy[nw], 0));
    }
    return GINT_OK;
}

int gint_launch_vlocal(gint_ctx* c, const double* V, double* H, cudaStream_t st, const double* V_host) {
    GINT_CUDA(cudaSetDevice(c->device));
    const size_t npts = (size_t)c->geom.N[0] * c->geom.N[1] * c->geom.N[2];
    if (c->n_values == 0) return GINT_OK;
    GINT_CUDA(cudaMemsetAsync(c->d_cval, 0, sizeof(double) * (size_t)c->n_cvalues, st));
    if (c->n_tiles > 0) {
        GINT_CUDA(cudaEventRecord(c->ev[0], st));
        int rc = launch_waves<true>(c, V, c->d_cval, st, V_host, nullptr);
        if (rc) return rc;
        GINT_CUDA(cudaEventRecord(c->ev[1], st));
        c->timed[0] = true;
    } else if (V_host) {
        GINT_CUDA(cudaMemcpyAsync(const_cast<double*>(V), V_host, sizeof(double) * npts, cudaMemcpyHostToDevice, st));
    }
    k_expand_H<<<(unsigned)((c->n_pairs + 7) / 8), 256, 0, st>>>(c->n_pairs, c->d_poff, c->d_pcanon, c->d_pflag, c->d_pnA, c->d_coff, c->d_cval, H);
    GINT_CUDA(cudaGetLastError());
    return GINT_OK;
}

int gint_launch_rho(gint_ctx* c, const double* D, double* rho, cudaStream_t st, double* rho_host) {
    GINT_CUDA(cudaSetDevice(c->device));
    const size_t npts = (size_t)(c->rho_planes > 0 ? std::min(c->rho_planes, c->geom.N[0]) : c->geom.N[0]) * c->geom.N[1] * c->geom.N[2];
    GINT_CUDA(cudaMemsetAsync(rho, 0, sizeof(double) * npts, st));
    if (c->n_tiles == 0) {
        if (rho_host) GINT_CUDA(cudaMemcpyAsync(rho_host, rho, sizeof(double) * npts, cudaMemcpyDeviceToHost, st));
        return GINT_OK;
    }
    k_sym_D<<<(unsigned)((c->n_canon + 7) / 8), 256, 0, st>>>(c->n_canon, c->d_poff, c->d_cpub, c->d_cmir, c->d_pnA, c->d_coff, D, c->d_cval);
    GINT_CUDA(cudaGetLastError());
    GINT_CUDA(cudaEventRecord(c->ev[2], st));
    int rc = launch_waves<false>(c, c->d_cval, rho, st, nullptr, rho_host);
    if (rc) return rc;
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

// ---------------------------------------------------------------------------------------------------
// FP64 peak micro-benchmark (gint_fp64_peak): registers only, 4 warps per SM sub-partition, 4 independent chains per warp.
template <bool MMA>
__global__ void __launch_bounds__(512) k_fp64_peak(int iters, double seed, double* __restrict__ sink, long long* __restrict__ ticks) {
    double c[4][2], f[16];
    const double a = seed + 1e-9 * threadIdx.x, b = 1.0 - seed;
    for (int i = 0; i < 4; i++) { c[i][0] = 0.0; c[i][1] = 0.0; }
    for (int i = 0; i < 16; i++) f[i] = a * i;
    const long long t0 = clock64();
    for (int it = 0; it < iters; it++) {
        if (MMA) {
#pragma unroll
            for (int r = 0; r < 4; r++)
#pragma unroll
                for (int i = 0; i < 4; i++)
                    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};" : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
        } else {
#pragma unroll
            for (int r = 0; r < 8; r++)
#pragma unroll
                for (int i = 0; i < 16; i++) f[i] = fma(f[i], a, b);
        }
    }
    const long long t1 = clock64();
    double s = 0.0;
    for (int i = 0; i < 4; i++) s += c[i][0] + c[i][1];
    for (int i = 0; i < 16; i++) s += f[i];
    if (s == 0.123456789) sink[0] = s;          // never true: keeps the loops alive
    if (blockIdx.x == 0 && threadIdx.x == 0) ticks[0] = t1 - t0;
}

extern "C" int gint_fp64_peak(int device, double out[4]) {
    if (!out) GINT_FAIL(GINT_ERR_INVALID_ARG, "out is NULL");
    DeviceGuard guard;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) GINT_FAIL(GINT_ERR_CUDA, "no usable CUDA device %d", device);
    GINT_CUDA(cudaSetDevice(device));
    cudaDeviceProp prop;
    GINT_CUDA(cudaGetDeviceProperties(&prop, device));
    const int nsm = prop.multiProcessorCount;
    double* d_sink = nullptr; long long* d_ticks = nullptr;
    GINT_CUDA(cudaMalloc(&d_sink, sizeof(double)));
    GINT_CUDA(cudaMalloc(&d_ticks, sizeof(long long)));
    cudaEvent_t e0, e1;
    GINT_CUDA(cudaEventCreate(&e0)); GINT_CUDA(cudaEventCreate(&e1));
    const int iters = 20000;
    for (int mode = 0; mode < 2; mode++) {
        float ms = 0.f;
        for (int rep = 0; rep < 2; rep++) {         // the first run warms up
            cudaEventRecord(e0, 0);
            if (mode == 0) k_fp64_peak<true><<<nsm, 512>>>(iters, 0.25, d_sink, d_ticks);
            else k_fp64_peak<false><<<nsm, 512>>>(iters, 0.25, d_sink, d_ticks);
            cudaEventRecord(e1, 0);
            if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d_sink); cudaFree(d_ticks); GINT_FAIL(GINT_ERR_CUDA, "gint_fp64_peak: %s", cudaGetErrorString(cudaGetLastError())); }
            cudaEventElapsedTime(&ms, e0, e1);
        }
        // per warp and iteration: 16 DMMAs of 8 x 8 x 4 multiply-adds / 128 fma instructions of 32 lanes
        const double fma_count = (double)nsm * 16.0 * iters * (mode == 0 ? 16.0 * 256.0 : 128.0 * 32.0);
        out[mode] = 2.0 * fma_count / (ms * 1e-3) / 1e12;
        if (mode == 0) {
            long long ticks = 0;
            cudaMemcpy(&ticks, d_ticks, sizeof(ticks), cudaMemcpyDeviceToHost);
            out[2] = (double)ticks / (ms * 1e-3) / 1e6;
        }
    }
    out[3] = nsm;
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d_sink); cudaFree(d_ticks);
    return GINT_OK;
}
