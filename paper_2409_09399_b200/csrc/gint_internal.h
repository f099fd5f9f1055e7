// gint_internal.h -- context layout and helpers shared by the translation units of libgint.so.
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>

#include "../../include/gint.h"

#define GINT_MAX_SHELL 12          // radial shells per species
#define GINT_MAX_NB 96             // neighbouring atom images per grid batch
#define GINT_MAX_GROUPS 32         // atom groups per batch (96 atoms of <= 32 orbitals in groups of <= 104 orbitals)
#define GINT_MAX_BS 8              // largest grid-batch edge along a1, a2 (points)
#define GINT_CZ 2                  // cubelet = 2 x 2 x 2 mesh points = the 8 columns of one DMMA operand pair
#define GINT_NCZ 8                 // a batch is at most 4 x 4 x GINT_NCZ cubelets: one 128-bit activity mask
#define GINT_CPTS 8                // points per cubelet
#define GINT_NCUB (16 * GINT_NCZ)  // cubelets per batch (at most 128)
#define GINT_MAX_BSZ (GINT_NCZ * GINT_CZ) // largest grid-batch edge along a3
// tile geometry of the contraction kernels: one tile = the block of H (or D) between two groups of atoms of one batch
#define GINT_TILE_ATOMS 8          // atom images per group
#define GINT_TILE_ORB 104          // orbitals per group = 13 fragments of 8 (8 atoms x 13 orbitals exactly)
#define GINT_TILE_FRAG 13
#define GINT_SEG_COLS 7            // column fragments of one segment
#ifndef GINT_MMA_WARPS
#define GINT_MMA_WARPS 12          // warp groups 0,1,2: DMMA consumers, three per SM sub-partition; each owns up to GINT_WARP_BLOCKS blocks
#endif
                                   // of 2 row fragments x 4 (block 0) or 3 (blocks 1, 2) column fragments of the tile
#ifndef GINT_WARP_BLOCKS
#define GINT_WARP_BLOCKS 3
#endif
#define GINT_AUX_WARPS 4           // warp group 3: warp 12 = TMA issuer, warps 13, 14 = reducers of gint_rho, warp 15 idle (setmaxnreg works on whole warp groups)
#define GINT_CTA_THREADS (32 * (GINT_MMA_WARPS + GINT_AUX_WARPS))
#ifndef GINT_REGS_MMA
#define GINT_REGS_MMA 152          // registers per thread after setmaxnreg: 384 * 152 + 128 * 56 = 65536
#endif
#ifndef GINT_REGS_AUX
#define GINT_REGS_AUX 56
#endif
// orbital values ("Phi") in global memory: one SLOT per (atom group, active cubelet) = [orbital row][8 points] doubles,
// rows padded to whole fragments, followed by one SIGN ROW (+-0.0 per point: the sign of V there; written by gint_vlocal only).
// 64 bytes per row = the unit of all Phi offsets
#define GINT_ROW_BYTES 64
#define GINT_SLOT_MAX_BYTES ((GINT_TILE_ORB + 1) * GINT_ROW_BYTES)   // 6720
// shared-memory ring of the contraction kernels: a stage = GINT_SC cubelets x (slot of group I, slot of group J)
#define GINT_SC 2
#ifndef GINT_NS
#define GINT_NS 7
#endif
#define GINT_STAGE_BYTES (GINT_SC * 2 * GINT_SLOT_MAX_BYTES)   // 26880
#define GINT_NCTX 4                // tile plans in flight per CTA (the issuer requests them ahead of the consumers)
#define GINT_PLAN_THREADS 96       // k_plan_fill (gint_init)
#define GINT_EVAL_THREADS 256      // orbital-evaluation kernel
#define GINT_TUNE_BATCHES 4096     // batches (of the largest shape) in the slab the batch-shape tuner times
#define GINT_TUNE_REPS 3            // timed runs per candidate shape (after one warm-up run); the least time counts
#define GINT_TUNE_MARGIN 0.02      // a shape replaces the default 8 x 8 x 16 only if it is this much faster (fraction)

// ---- error plumbing -------------------------------------------------------------------------------
void gint_set_error(const char* fmt, ...);
#define GINT_FAIL(code, ...) do { gint_set_error(__VA_ARGS__); return (code); } while (0)
#define GINT_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { \
    gint_set_error("%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
    return e_ == cudaErrorMemoryAllocation ? GINT_ERR_OUT_OF_MEMORY : GINT_ERR_CUDA; } } while (0)

// The entry points run on the context's device and give the caller's current device back on return.
struct DeviceGuard {
    int prev = -1;
    DeviceGuard() { if (cudaGetDevice(&prev) != cudaSuccess) prev = -1; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// ---- device-side descriptions ---------------------------------------------------------------------
struct SpeciesDev {
    double rc;                      // cutoff radius
    int n_shell;
    int norb;
    int n_int;                      // spline intervals per shell (n_knot - 1)
    int tab_off;                    // first cell (double2) of this species in the radial table
    int row_len;                    // cells per knot = n_shell
    int l[GINT_MAX_SHELL];
};

// Geometry and batching constants, passed by value to every kernel.
struct Geom {
    double a[9];                    // cell rows a1,a2,a3
    double inv[9];                  // frac = pos * inv (row vector convention)
    double hgt[3];                  // distance between lattice planes along each axis
    double step[9];                 // mesh steps: rows a1/N1, a2/N2, a3/N3
    double dV;
    double inv_dr;
    int N[3];                       // mesh
    int bs[3];                      // batch edge lengths (points)
    int nb[3];                      // batches along each axis
    int K;                          // bs[0]*bs[1]*bs[2]
    int key_m;                      // pair keys: |n_i| <= key_m, key_M = 2*key_m+1
    int key_M;
    int max_cols;                   // max orbitals of one batch
    int max_nb;                     // max neighbour entries of one batch
};

// One neighbouring atom image of a grid batch.
struct NeighEntry {
    int atom;
    int shift;                      // (t1+64) | (t2+64)<<8 | (t3+64)<<16
    unsigned long long mask[2];     // bit ((cx*4 + cy)*GINT_NCZ + cz) of the 128: cubelet of the batch with a point inside the sphere
};

__host__ __device__ inline int pack_shift(int t1, int t2, int t3) { return (t1 + 64) | ((t2 + 64) << 8) | ((t3 + 64) << 16); }
__host__ __device__ inline void unpack_shift(int s, int& t1, int& t2, int& t3) {
    t1 = (s & 255) - 64; t2 = ((s >> 8) & 255) - 64; t3 = ((s >> 16) & 255) - 64;
}

// Mesh point (i,j,k) -> Cartesian position (reading R1).  Used by the neighbour pass AND the orbital
// evaluation so that both take the |d| < rc decision on bit-identical numbers.
__host__ __device__ inline void mesh_point(const Geom& g, int i, int j, int k, double& x, double& y, double& z) {
    const double u = (double)i, v = (double)j, w = (double)k;
    x = fma(w, g.step[6], fma(v, g.step[3], u * g.step[0]));
    y = fma(w, g.step[7], fma(v, g.step[4], u * g.step[1]));
    z = fma(w, g.step[8], fma(v, g.step[5], u * g.step[2]));
}

// Position of atom image (A, t): tau_A + t1 a1 + t2 a2 + t3 a3, with explicit fma so that host and device agree bit by bit
// (the neighbour pass, the activity masks and the orbital evaluation all take the |d| < rc decision on these numbers).
__host__ __device__ inline void image_pos(const Geom& g, const double* p, int t1, int t2, int t3, double& x, double& y, double& z) {
    const double u = (double)t1, v = (double)t2, w = (double)t3;
    x = fma(w, g.a[6], fma(v, g.a[3], fma(u, g.a[0], p[0])));
    y = fma(w, g.a[7], fma(v, g.a[4], fma(u, g.a[1], p[1])));
    z = fma(w, g.a[8], fma(v, g.a[5], fma(u, g.a[2], p[2])));
}

// ---- tile plans -----------------------------------------------------------------------------------
// Everything the contraction kernels need to know about one tile = (batch, atom group I, atom group J) depends on the geometry
// only.  gint_init writes it once per tile into a PLAN in global memory; at run time the issuer warp of a persistent CTA fetches
// the plan of its next tile with one TMA bulk copy.  Layout: PlanHdr, then ncub + GINT_SC records PlanCub (the last GINT_SC
// are zero: the consumers prefetch one stage ahead), padded to a multiple of 16 bytes.
struct PairEnt { unsigned off; unsigned short sr, sc; };   // element (oa, ob) of the atom pair at off + oa*sr + ob*sc (canonical value array); off = ~0u: none
struct alignas(16) PlanHdr {
    int valid;                          // 0: the queue is empty, the roles leave (written by the issuer, never stored)
    int ncub, nstage;                   // cubelets the tile walks over; ring stages of GINT_SC cubelets
    int zero;                           // always 0: the consumers' opaque loop condition (keeps ptxas from predicating the DMMA blocks)
    int nI, nJ, nfI, nfJ;               // atoms / fragments of the two groups
    int RI, RJ, diag, pad0;             // orbital rows (padded to fragments); I == J
    int i0, j0, k0, pad1;               // batch origin (mesh points)
    int ex, ey, ez, pad2;               // batch extents (mesh points; ragged at the mesh edge)
    unsigned long long rowI, rowJ;      // first 64-byte row of the two groups' slot arrays (numbering over the whole mesh)
    unsigned blk[GINT_WARP_BLOCKS][GINT_MMA_WARPS];   // consumer warp w, block k: first row fragment | second row present << 4 | first column
                                        // fragment << 5 | n column fragments << 9   (n = 0: unused).  Block 0 holds up to 4 columns, blocks 1, 2 up to 3.
    PairEnt pair[GINT_TILE_ATOMS][GINT_TILE_ATOMS];   // canonical block of (I atom a, J atom b)
    unsigned char row_atom[2][GINT_TILE_ORB];   // orbital row -> atom slot inside the group (255 = padding)
    unsigned char row_orb[2][GINT_TILE_ORB];    // orbital row -> orbital index inside the atom
};
struct PlanCub {                        // one listed cubelet
    unsigned short slotI, slotJ;        // its slot inside the two groups' slot arrays
    unsigned char cub, pad[3];          // its bit number in the batch's activity masks
    unsigned char vis[16];              // per consumer warp: bits 2k, 2k+1 = rows of the warp's block k to work on there (0: skip)
};
static_assert(sizeof(PlanHdr) % 16 == 0 && sizeof(PlanCub) == 24, "plan layout");
#define GINT_PLAN_MAX_BYTES ((sizeof(PlanHdr) + (GINT_NCUB + GINT_SC + 1) * sizeof(PlanCub) + 15) & ~(size_t)15)
__host__ __device__ inline unsigned plan_units(int ncub) { return (unsigned)((sizeof(PlanHdr) + (size_t)(ncub + GINT_SC) * sizeof(PlanCub) + 15) >> 4); }   // 16-byte units

struct gint_ctx {
    int device = 0;
    Geom geom{};
    // basis
    int n_species = 0;
    std::vector<SpeciesDev> h_species;
    SpeciesDev* d_species = nullptr;
    double* d_tab = nullptr;         // cells {y, y'' dr^2/6}: [species][knot][shell]
    size_t tab_bytes = 0;
    bool tab_in_smem = false;        // the contraction kernels copy the table into shared memory
    // atoms
    int n_atoms = 0;
    std::vector<int> h_atom_species;
    std::vector<double> h_atom_pos;
    double* d_atom_pos = nullptr;    // [n_atoms*3]
    int* d_atom_species = nullptr;
    long long n_orb_total = 0;
    // public pair list (lexicographic), host copies for gint_get_pairs
    long long n_pairs = 0, n_values = 0;
    std::vector<int> h_pA, h_pB, h_pR;
    std::vector<long long> h_poff;
    long long* d_poff = nullptr;     // [n_pairs+1] offsets of the public blocks
    int* d_pcanon = nullptr;         // [n_pairs] canonical index of the key itself or of its mirror
    unsigned char* d_pflag = nullptr;// [n_pairs] 1 = key is canonical, 0 = key is the mirror of a canonical key
    int* d_pnA = nullptr;            // [n_pairs] norb(A) | norb(B) << 16
    // canonical (one per mirror pair) keys: the internal accumulation layout
    long long n_canon = 0, n_cvalues = 0;
    int* d_crow = nullptr;           // [n_atoms+1] first canonical key of row A
    unsigned long long* d_ckey = nullptr; // [n_canon] packed (B, n) ascending inside a row
    unsigned int* d_coff = nullptr;  // [n_canon+1] offsets (doubles) into the canonical value array
    int* d_cpub = nullptr;           // [n_canon] public index of the canonical key
    int* d_cmir = nullptr;           // [n_canon] public index of its mirror (== d_cpub for (A,A,0))
    double* d_cval = nullptr;        // [n_cvalues] canonical-half scratch: H accumulation / symmetrised D
    // batches
    long long n_batch_total = 0, n_batch = 0, n_batch_empty = 0, n_entries = 0;
    int* d_bstart = nullptr;         // [n_batch_total+1] CSR into d_bent
    NeighEntry* d_bent = nullptr;    // neighbour entries sorted by (atom, shift lexicographic)
    long long n_tiles = 0;
    int2* d_tile = nullptr;          // [n_tiles] {batch id, I | J<<8 | G<<16}: group pair (I <= J) of G groups of the batch (freed once the plans exist)
    unsigned* d_planoff = nullptr;   // [n_tiles+1] offsets of the tile plans in 16-byte units
    unsigned char* d_plan = nullptr; // tile plans
    size_t plan_bytes = 0;
    int* d_tstart = nullptr;         // [n_batch_total+1] first tile of each batch
    int* d_gstart = nullptr;         // [n_batch_total+1] first atom group of each batch (CSR into d_goff)
    unsigned long long* d_goff = nullptr; // [sum G] Phi offset (rows of 64 bytes, whole mesh) of each (batch, group) slot array
    // waves: contiguous batch ranges whose orbital values fit the Phi scratch buffer
    struct Wave { long long b0, b1, t0, t1; unsigned long long row0, rows; };
    std::vector<Wave> waves;
    double* d_phi = nullptr;         // Phi scratch of one wave
    size_t phi_bytes = 0;
    unsigned long long phi_rows_total = 0;
    int* d_queue = nullptr;          // [waves] tile-queue heads
    int n_sm = 0;
    long long padded_macs = 0;
    size_t smem_bytes = 0;           // contraction kernels
    size_t smem_eval = 0;            // evaluation kernel
    size_t device_bytes = 0;
    size_t device_bytes_base = 0;    // before the batch structures (the tuner builds and frees several of them)
    // batch-shape tuner (GINT_FLAG_TUNE): what was tried
    struct TuneResult { int bs[3]; double ns_per_point; };
    std::vector<TuneResult> tune;
    double tune_seconds = 0.0;
    // lazily computed statistics
    bool have_alg = false;
    long long alg[4] = {0, 0, 0, 0};
    // CUDA events around the two main kernels (gint_kernel_times)
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    bool timed[2] = {false, false};
    // per-wave events (gint_phase_times): [call][2 * wave] after the evaluation kernel, [call][2 * wave + 1] after the tile kernel
    std::vector<cudaEvent_t> ev_wave[2];
    // host-path staging; the copies run on a stream of their own, chunk by chunk beside the waves
    double* d_stage_in = nullptr; size_t stage_in_n = 0;
    double* d_stage_out = nullptr; size_t stage_out_n = 0;
    cudaStream_t copy_stream = nullptr;
    size_t smem_optin = 0;           // cudaDevAttrMaxSharedMemoryPerBlockOptin of the device (set by gint_init)
    bool want_force = false;         // GINT_FLAG_FORCE: the batch shape must also fit the force kernel's shared memory
    bool force_configured = false;   // k_force_batch's shared-memory limit has been raised on this context's device
    int rho_planes = 0;              // > 0 (batch-shape tuner only): gint_rho clears just the first rho_planes mesh planes along a1
    // gint_force_stress: full-layout copy of D + mirror^T (allocated by the first call), events around its kernels
    double* d_dfull = nullptr;
    cudaEvent_t ev_force[2] = {nullptr, nullptr};
    bool timed_force = false;
    std::vector<cudaEvent_t> ev_copy;  // [waves + 1]
};

// implemented in gint_kernels.cu
// V_host / rho_host (optional): the host buffer behind V (gint_vlocal) or in front of rho (gint_rho); the copies then run in chunks,
// one per wave, on the context's copy stream beside the kernels
int gint_launch_vlocal(gint_ctx* c, const double* V, double* H, cudaStream_t st, const double* V_host = nullptr);
int gint_launch_rho(gint_ctx* c, const double* D, double* rho, cudaStream_t st, double* rho_host = nullptr);
int gint_launch_alg_stats(gint_ctx* c);
int gint_launch_force(gint_ctx* c, const double* V, const double* D, double* F, double* sigma, cudaStream_t st);   // gint_force.cu
size_t gint_force_smem(const gint_ctx* c);
int gint_configure_kernels(gint_ctx* c);
size_t gint_smem_needed(gint_ctx* c, size_t limit);   // also decides tab_in_smem
int gint_build_phi_layout(gint_ctx* c, const int* d_bgroups, size_t phi_cap_bytes, bool* batch_too_big);   // Phi offsets of every (batch, group), waves, scratch
int gint_build_plans(gint_ctx* c);                    // tile plans (after the Phi layout)
int gint_device_excl_scan(const int* d_in, long long n, int* d_out, long long* total);   // gint_init.cu

// Split of the n neighbour entries of a batch into G groups of consecutive entries: group k = [k*n/G, (k+1)*n/G).
__host__ __device__ inline int group_begin(int k, int n, int G) { return (int)(((long long)k * n) / G); }
