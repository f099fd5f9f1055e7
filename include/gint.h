/*
 * gint.h -- C ABI of libgint.so: real-space grid integration for numerical-atomic-orbital (LCAO)
 * Kohn-Sham DFT on one NVIDIA B200 (sm_100a), fp64.
 *
 * What the library computes (PAPER.md = arXiv 2409.09399 text, /root/reference/PAPER.md):
 *   gint_vlocal  Eq. 2:  H_{mu nu} = sum_r phi_mu(r - R_mu) V(r) phi_nu(r - R_nu) dV
 *   gint_rho     Eq. 3:  rho(r)    = sum_{mu nu} rho_{mu nu} phi_mu(r - R_mu) phi_nu(r - R_nu)
 *   on a uniform periodic mesh, processed in grid batches whose "neighbouring atoms" are the atoms with a
 *   batch point closer than their cutoff radius (section 2.3.2); orbitals are
 *   zero at and beyond the cutoff (Fig. 6).
 * Conventions the paper leaves open are fixed in DESIGN.md "Readings" (R1..R9) and repeated at each call.
 *
 * General rules
 *   - every function returns GINT_OK (0) or a negative gint_status; none throws or exits;
 *     gint_last_error() returns a thread-local, NUL-terminated message for the last failure.
 *   - units: bohr.  All host arrays are BORROWED for the duration of the call and copied inside.
 *   - device pointers are BORROWED, must be 8-byte aligned and belong to the device given to gint_init.
 *   - gint_vlocal / gint_rho only ENQUEUE work on the given CUDA stream (a cudaStream_t passed as void*,
 *     e.g. torch.cuda.current_stream().cuda_stream); they do not synchronise.  A context owns its
 *     neighbour tables and scratch buffers: do not use one context from two streams at the same time.
 *   - there is no CPU fallback: without a usable CUDA device gint_init fails with GINT_ERR_CUDA.
 */
#ifndef GINT_H
#define GINT_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gint_ctx gint_ctx;

typedef enum gint_status {
    GINT_OK = 0,
    GINT_ERR_INVALID_ARG = -1,   /* NULL pointer, negative size, non-finite value, det(cell) <= 0, ...        */
    GINT_ERR_UNSUPPORTED = -2,   /* l > 2, more than GINT_MAX_ORB orbitals per atom, batch edge too large, device not sm_100 */
    GINT_ERR_CUDA = -3,          /* a CUDA runtime call failed (message holds cudaGetErrorString)             */
    GINT_ERR_OUT_OF_MEMORY = -4, /* host or device allocation failed                                          */
    GINT_ERR_BAD_STATE = -5      /* NULL / freed context                                                      */
} gint_status;

#define GINT_MAX_L 2
#define GINT_MAX_ORB 32          /* orbitals per atom (sum over shells of 2l+1) */

/* flags of gint_init: three 8-bit fields override the grid-batch edge lengths (mesh points) along a1,a2,a3: 1..8, 1..8, 1..16;
 * 0 = choose automatically: 8x8x16 points, or the largest smaller shape whose batches have at most 96 neighbouring atom
 * images (PAPER.md:165 uses batches of 27..1000 points; Table 3 sweeps 125..512).  A larger edge is GINT_ERR_UNSUPPORTED. */
/* GINT_FLAG_TUNE (with no batch-edge field set): gint_init times gint_vlocal + gint_rho for several grid-batch shapes on a slab of the
 * mesh of fixed size (the paper's online auto-tuning; there over GEMM tile sizes, here over the grid-batch shape,
 * the parameter its Table 3 sweeps by hand).  Each shape's time is the least of three runs after a warm-up run.  The default
 * 8x8x16 is kept unless the fastest other shape beats it by more than 2 %, so that timing noise does not flip the choice (and with
 * it memory use and summation order) from run to run.  A shape that cannot be built or run is skipped (reported as -1); if the
 * tuner's own buffers (two slabs of the mesh, 2 * n_values doubles) cannot be allocated, gint_init goes on untuned instead of failing.
 * gint_tune_report tells what was tried. */
#define GINT_FLAG_TUNE (1ull << 32)
/* GINT_FLAG_PHI_CAP_MB(mb), mb = 1..1048575: upper bound, in MiB, of the context's orbital-value scratch (the buffer one "wave" of grid
 * batches is evaluated into before it is contracted; GINT_STAT_PHI_SCRATCH_BYTES, GINT_STAT_N_WAVES).  0 = automatic: the smaller of
 * 16 GiB and a quarter of the device memory free at gint_init.  A smaller cap trades memory for more, shorter waves; a batch shape
 * whose single largest batch exceeds the cap counts as "does not fit" and the next smaller shape is tried. */
#define GINT_FLAG_PHI_CAP_MB(mb) (((unsigned long long)(mb) & 0xfffffull) << 40)
/* GINT_FLAG_FORCE: the context will be used for gint_force_stress as well.  The force kernel keeps the orbital values and the
 * Psi rows of a whole batch in shared memory, so it can need more of it than the contraction kernels; with this flag the automatic
 * choice of the batch shape (and the tuner) only accepts shapes that gint_force_stress supports too.  Without it gint_force_stress
 * may return GINT_ERR_UNSUPPORTED on cells with many orbitals per batch although gint_vlocal / gint_rho work. */
#define GINT_FLAG_FORCE (1ull << 33)
#define GINT_FLAG_BATCH(bx, by, bz) ((unsigned long long)(bx) | ((unsigned long long)(by) << 8) | ((unsigned long long)(bz) << 16))

/*
 * gint_init -- "gint_init(basis tables, atoms, cell, mesh)" of BASELINE.json north_star.
 * Builds, on the device: the radial interpolation tables, the sparse pair list (all ordered keys
 * (A, B, n) with |tau_B + n.cell - tau_A| < rc_A + rc_B, strict; reading R7), the grid batches and, per
 * batch, the list of atom images with at least one batch point closer than rc.
 *
 *   n_species, n_shell[n_species], shell_l[sum n_shell] (0..2), rcut[n_species] (bohr)
 *   dr                    radial table spacing; knot i of every shell sits at r = i*dr
 *   n_knot[n_species]     knots per shell of that species; (n_knot-1)*dr must be >= rcut
 *   tab_y, tab_y2         concatenated [species][shell][knot] radial values R(i*dr) and cubic-spline second
 *                         derivatives (input DATA; reading R5: R(r) = a y_i + b y_{i+1} + ((a^3-a) y2_i +
 *                         (b^3-b) y2_{i+1}) dr^2/6 with i = min(floor(r/dr), n_knot-2), b = r/dr - i, a = 1-b)
 *   n_atoms, atom_species[n_atoms], atom_pos[n_atoms*3]   Cartesian, need not be wrapped into the cell
 *   cell[9]               rows a1, a2, a3; det > 0
 *   mesh[3]               N1, N2, N3 >= 1; mesh point (i,j,k) sits at (i/N1) a1 + (j/N2) a2 + (k/N3) a3,
 *                         flat index g = (i*N2 + j)*N3 + k, dV = det(cell)/(N1 N2 N3)            (reading R1)
 *   device                CUDA device ordinal
 * Orbital of shell s, m = -l..l:  phi = R_s(|d|) Y_lm(d/|d|), d = r - tau_A - n.cell, zero for |d| >= rc;
 * real spherical harmonics without Condon-Shortley phase, order l=1: (y,z,x), l=2: (xy,yz,3z^2-1,xz,x^2-y^2)
 * (reading R4).  Orbitals of one atom are ordered by shell, then m.
 * On success *out owns device memory until gint_free.
 */
int gint_init(gint_ctx** out,
              int n_species, const int* n_shell, const int* shell_l, const double* rcut,
              double dr, const int* n_knot, const double* tab_y, const double* tab_y2,
              int n_atoms, const int* atom_species, const double* atom_pos,
              const double cell[9], const int mesh[3],
              int device, unsigned long long flags);

/* total orbitals = sum over atoms of norb(species). */
int gint_n_orb(const gint_ctx* ctx, long long* n_orb_total);

/* number of ordered pair keys and total doubles of an H (or D) value array. */
int gint_n_pairs(const gint_ctx* ctx, long long* n_pairs, long long* n_values);

/* pair list in lexicographic order of (A, B, n1, n2, n3): A[n_pairs], B[n_pairs], R3[n_pairs*3],
 * offset[n_pairs+1] (host arrays supplied by the caller; any may be NULL to skip).  Block p is row-major
 * norb(A) x norb(B) doubles at offset[p].  Both (A,B,n) and (B,A,-n) are listed. */
int gint_get_pairs(const gint_ctx* ctx, int* A, int* B, int* R3, long long* offset);

/*
 * gint_vlocal -- Eq. 2 made periodic (reading R8):
 *   H_p[mu,nu] = dV * sum_g V_g * sum_{t in Z^3} phi_{A mu}(r_g; t) phi_{B nu}(r_g; t + n),   p = (A,B,n).
 *   V_dev  device, N1*N2*N3 doubles, index g (N3 fastest)           -- read
 *   H_dev  device, n_values doubles in pair-list layout               -- OVERWRITTEN (every block, both
 *          (A,B,n) and its mirror (B,A,-n) = transpose)
 */
int gint_vlocal(gint_ctx* ctx, const double* V_dev, double* H_dev, void* cuda_stream);

/*
 * gint_rho -- Eq. 3, reading R9:
 *   rho_g = sum over ordered pairs of atom images ((A,t),(B,t')) non-zero at r_g of
 *           phi_A(r_g;t)^T  D_(A,B,t'-t)  phi_B(r_g;t').      No symmetry of D is assumed.
 *   D_dev    device, n_values doubles in pair-list layout             -- read
 *   rho_dev  device, N1*N2*N3 doubles                                 -- OVERWRITTEN
 */
int gint_rho(gint_ctx* ctx, const double* D_dev, double* rho_dev, void* cuda_stream);

/* Eq. 4 and Eq. 5: Pulay force and stress of the local-potential energy E = <D, H> = dV sum_g V_g rho_g, at fixed V
 * (per mesh index), D and dV (reading R15 of DESIGN.md; orbital gradients: spline derivative and gradient of the real harmonics,
 * PAPER.md:163):
 *   F_C^a      = -dE/dtau_C^a      = dV sum_g V_g sum_t grad_a phi_(C,t)(r_g) . Psi_(C,t)(r_g),
 *   Psi_(C,t)  = sum over atom images (B,t') non-zero at r_g of ( D_(C,B,t'-t) + D_(B,C,t-t')^T ) phi_(B,t')(r_g),
 *   sigma^{ab} = -(1/Omega) dE/d eps_ab = -(1/Omega) sum_(C,t) dV sum_g V_g ( grad_a phi . Psi ) (r_g - tau_C - t)^b
 * (the factor 1/Omega that Eq. 4 prints for the force is dropped; tau^b of Eq. 5 is read relative to the integration point).
 * No symmetry of D is assumed.
 *   V_dev     device, N1*N2*N3 doubles                                 -- read
 *   D_dev     device, n_values doubles in pair-list layout             -- read
 *   F_dev     device, 3 * n_atoms doubles, [atom][x, y, z]             -- OVERWRITTEN
 *   sigma_dev device, 9 doubles [a][b], or NULL (stress not wanted)    -- OVERWRITTEN
 * Enqueued on `cuda_stream`, no synchronisation.  The first call allocates a context-owned copy of D in the pair-list layout
 * (8 * n_values bytes; GINT_ERR_OUT_OF_MEMORY if that fails).  GINT_ERR_UNSUPPORTED: more than 2^32 matrix elements, or a
 * grid batch that does not fit the kernel's shared memory: about 8.6 KB + 4 n^2 + 192 n + 128 R bytes for the n atom images and R
 * orbitals of the largest batch, against 227 KB per CTA (R <= about 1,300 at n = 96, 1,600 at n = 32).  GINT_FLAG_FORCE at
 * gint_init picks a batch shape that fits. */
int gint_force_stress(gint_ctx* ctx, const double* V_dev, const double* D_dev, double* F_dev, double* sigma_dev, void* cuda_stream);

/*
 * gint_force_stress_static -- gint_force_stress for callers that cannot allocate device memory.
 *
 * Who needs it: a host code that gave the whole GPU to its own memory arena at start-up (so a cudaMalloc inside a library fails),
 * a process confined to a fixed MPS / MIG memory slice, or a relaxation loop that cannot tolerate the device-wide stall a
 * cudaMalloc / cudaFree may cause while its other streams are running.  gint_force_stress does one such allocation (its
 * 8 * n_values-byte symmetrised copy of D, on the first call); this variant keeps that copy in a fixed array that is part of the
 * library's own device image instead, and calls no cudaMalloc, cudaFree or other allocating routine.
 *
 * Same arguments, same result (to rounding: the floating-point atomics add in a different order from call to call) and same
 * errors as gint_force_stress, plus:
 *   - GINT_ERR_UNSUPPORTED when n_values (gint_n_pairs) exceeds GINT_STATIC_SCRATCH_DOUBLES; nothing is enqueued then.
 *     1,048,576 doubles = 8 MiB: enough for the 8-atom diamond and 72-atom graphene cells of the test suite (0.17 M / 0.82 M
 *     elements), not for the twisted-bilayer cells.  The array costs that much memory on every GPU that loads libgint.so, used or not.
 *   - The first call on a device looks up the array's device address and raises the kernel's shared-memory limit.  Make that first
 *     call outside any stream capture; later calls only enqueue two memsets, two kernels and two event records.
 *   - One array per device serves all contexts, streams and threads and keeps what the last call left in it.  The call rewrites the
 *     part it reads, so stale contents are harmless, but two calls that may overlap on the GPU race on it: put them on one stream
 *     (or order them with events).  gint_force_stress has its own per-context copy and may run beside this one.
 * gint_force_time reports this call's kernels as well.
 */
#define GINT_STATIC_SCRATCH_DOUBLES (1 << 20)
int gint_force_stress_static(gint_ctx* ctx, const double* V_dev, const double* D_dev, double* F_dev, double* sigma_dev, void* cuda_stream);

/* Device duration (seconds) of the kernels of the LAST gint_force_stress call (CUDA events on the caller's stream); -1 before it. */
int gint_force_time(gint_ctx* ctx, double* seconds);

/* Host-buffer convenience forms (the end-to-end path timed by bench.py's "e2e"): copy the input from host
 * memory (pinned or pageable) to context-owned device buffers, run the device path, copy the result back to
 * host memory and synchronise the stream before returning. */
int gint_vlocal_host(gint_ctx* ctx, const double* V_host, double* H_host, void* cuda_stream);
int gint_rho_host(gint_ctx* ctx, const double* D_host, double* rho_host, void* cuda_stream);

/* statistics, out[GINT_N_STATS] (long long).  Filled at init except the GINT_STAT_ALG_* entries, which are
 * counted on the device on the first call that asks for them (the context is not const for that reason). */
enum {
    GINT_STAT_N_BATCH = 0,        /* non-empty grid batches                                                 */
    GINT_STAT_N_BATCH_EMPTY = 1,  /* batches without any neighbouring atom                                  */
    GINT_STAT_BATCH_BX = 2, GINT_STAT_BATCH_BY = 3, GINT_STAT_BATCH_BZ = 4,
    GINT_STAT_NEIGH_ENTRIES = 5,  /* sum over batches of neighbouring atom images                          */
    GINT_STAT_MAX_NB = 6,         /* max neighbouring atom images of one batch                              */
    GINT_STAT_MAX_COLS = 7,       /* max orbitals of one batch                                              */
    GINT_STAT_PADDED_MACS = 8,    /* sum_b k_b * cols_b^2 (what a dense, non-symmetric batch product costs) */
    GINT_STAT_N_CANON = 9,        /* canonical pair keys (one of each mirror pair)                          */
    GINT_STAT_ALG_INCIDENCE = 10, /* sum_g #atoms with |d| < rc at g                                        */
    GINT_STAT_ALG_SUM_N = 11,     /* sum_g n_g,   n_g = orbitals non-zero at g                              */
    GINT_STAT_ALG_SUM_N2 = 12,    /* sum_g n_g^2                                                            */
    GINT_STAT_NONEMPTY_POINTS = 13,
    GINT_STAT_SMEM_BYTES = 14,    /* dynamic shared memory of the contraction kernels (TMA ring + tile contexts) */
    GINT_STAT_DEVICE_BYTES = 15,  /* device memory owned by the context                                     */
    GINT_STAT_LAUNCHES_VLOCAL = 16, /* kernels one gint_vlocal call launches (memsets not counted)          */
    GINT_STAT_LAUNCHES_RHO = 17,  /* kernels one gint_rho call launches                                     */
    GINT_STAT_SMEM_EVAL = 18,     /* dynamic shared memory of the orbital-evaluation kernel                 */
    GINT_STAT_TAB_IN_SMEM = 19,   /* 1: the evaluation kernel reads the radial table from shared memory     */
    GINT_STAT_PHI_BYTES = 20,     /* orbital values one call evaluates and writes (all waves), bytes        */
    GINT_STAT_PHI_SCRATCH_BYTES = 21, /* size of the context's orbital-value scratch buffer (one wave)      */
    GINT_STAT_N_WAVES = 22,       /* waves (evaluate + contract launches) per call                          */
    GINT_STAT_N_TILES = 23,       /* (batch, group pair) tiles per call                                     */
    GINT_STAT_TUNE_US = 24,       /* microseconds gint_init spent in the batch-shape tuner (0: not asked for) */
    GINT_N_STATS = 25
};
int gint_stats(gint_ctx* ctx, long long* out);

/* What the batch-shape tuner tried: up to max_rows rows of out[4] = {bx, by, bz, nanoseconds per mesh point of gint_vlocal + gint_rho
 * on the tuning slab, or -1 if the shape did not fit}; *n_rows = rows written (0 when gint_init ran without GINT_FLAG_TUNE). */
int gint_tune_report(const gint_ctx* ctx, int max_rows, double* out, int* n_rows);

/* Device durations (seconds) of the LAST gint_vlocal / gint_rho call on this context, between two CUDA events recorded on the
 * caller's stream: one before the first wave's orbital-evaluation kernel, one after the last wave's tile-contraction kernel.  The
 * span therefore covers the evaluation and contraction kernels of every wave and, for the *_host forms, the time the stream waits
 * for a wave's chunk of V to arrive; it leaves out the clearing memset, the symmetrisation of D (gint_rho) and the expansion of the
 * canonical blocks into H (gint_vlocal).  Synchronises on those events.  out[0] = gint_vlocal, out[1] = gint_rho; an entry is -1 when
 * that call has not been made yet. */
int gint_kernel_times(gint_ctx* ctx, double out[2]);

/* The same, split by kernel: out[0] / out[1] = orbital-evaluation kernels / tile-contraction kernels (summed over the waves) of the
 * last gint_vlocal call, out[2] / out[3] = of the last gint_rho call; -1 when that call has not been made yet. */
int gint_phase_times(gint_ctx* ctx, double out[4]);

/* FP64 peak of the device, measured now (the roofline denominator's cross-check): a register-only micro-benchmark
 * on all SMs, 16 warps per SM, timed with CUDA events on the default stream of `device`.
 *   out[0]  DMMA.8x8x4 (mma.sync.m8n8k4.f64, the instruction of the contraction kernels), TFLOP/s (2 flop per multiply-add)
 *   out[1]  DFMA (fma.rn.f64), TFLOP/s
 *   out[2]  SM clock during the DMMA run, MHz (clock64 ticks / elapsed time)
 *   out[3]  number of SMs
 * Synchronises the device.  GINT_ERR_CUDA without a usable device. */
int gint_fp64_peak(int device, double out[4]);

int gint_free(gint_ctx* ctx);

const char* gint_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GINT_H */
