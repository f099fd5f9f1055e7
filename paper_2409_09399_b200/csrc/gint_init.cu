// gint_init.cu -- context construction: radial coefficient tables, sparse pair list, grid batches and the
// per-batch neighbour lists (north_star step 1; PAPER.md:141, PAPER.md:153-155 describe the paper's host-side
// "sub-task" generation, which here runs once per geometry on the device and stays resident).
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdlib>
#include <cstring>
#include <new>
#include <chrono>

#include "gint_internal.h"

// ---------------------------------------------------------------------------------------------------
// error message (thread local)
static thread_local char g_err[512] = "";
void gint_set_error(const char* fmt, ...) {
    va_list ap; va_start(ap, fmt); vsnprintf(g_err, sizeof(g_err), fmt, ap); va_end(ap);
}
extern "C" const char* gint_last_error(void) { return g_err; }

// ---------------------------------------------------------------------------------------------------
// small device helpers
__device__ __forceinline__ int warp_incl_scan(int v) {
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { int t = __shfl_up_sync(0xffffffffu, v, d); if (lane >= d) v += t; }
    return v;
}
// exclusive scan over a 256-thread block; returns the exclusive prefix, writes the block total.
__device__ int block_excl_scan_256(int v, int* s_warp /*[9]*/, int& total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int inc = warp_incl_scan(v);
    __syncthreads();
    if (lane == 31) s_warp[w] = inc;
    __syncthreads();
    if (w == 0) {
        int x = lane < 8 ? s_warp[lane] : 0;
        int xi = warp_incl_scan(x);
        if (lane < 8) s_warp[lane] = xi - x;
        if (lane == 7) s_warp[8] = xi;
    }
    __syncthreads();
    total = s_warp[8];
    return inc - v + s_warp[w];
}

// ---------------------------------------------------------------------------------------------------
// Pair keys (reading R7): all ordered (A, B, n) with |tau_B + n.cell - tau_A| < rc_A + rc_B, strict,
// lexicographic in (A, B, n1, n2, n3).  One CTA per A; threads take consecutive B; ordered compaction.
template <bool FILL>
__global__ void __launch_bounds__(256) k_pairs(Geom g, int n_atoms, const double* __restrict__ pos, const int* __restrict__ spec,
                                               const SpeciesDev* __restrict__ sp, int* __restrict__ row_count,
                                               const long long* __restrict__ row_start, int* __restrict__ pB, int* __restrict__ pR) {
    __shared__ int s_warp[9];
    const int A = blockIdx.x;
    const double ax = pos[3 * A], ay = pos[3 * A + 1], az = pos[3 * A + 2];
    const double rcA = sp[spec[A]].rc;
    long long running = 0;
    for (int B0 = 0; B0 < n_atoms; B0 += 256) {
        const int B = B0 + threadIdx.x;
        int cnt = 0;
        int lo[3] = {0, 0, 0}, hi[3] = {-1, -1, -1};
        double dx = 0, dy = 0, dz = 0, rmax = 0;
        if (B < n_atoms) {
            dx = pos[3 * B] - ax; dy = pos[3 * B + 1] - ay; dz = pos[3 * B + 2] - az;
            rmax = rcA + sp[spec[B]].rc;
            for (int i = 0; i < 3; i++) {
                double f = dx * g.inv[i] + dy * g.inv[3 + i] + dz * g.inv[6 + i];
                double ext = rmax / g.hgt[i];
                lo[i] = (int)floor(-f - ext) - 1 + 1;     // ceil(-f-ext) >= floor(-f-ext); keep one spare on each side
                hi[i] = (int)ceil(-f + ext);
            }
            for (int n1 = lo[0]; n1 <= hi[0]; n1++) for (int n2 = lo[1]; n2 <= hi[1]; n2++) for (int n3 = lo[2]; n3 <= hi[2]; n3++) {
                double x = dx + n1 * g.a[0] + n2 * g.a[3] + n3 * g.a[6];
                double y = dy + n1 * g.a[1] + n2 * g.a[4] + n3 * g.a[7];
                double z = dz + n1 * g.a[2] + n2 * g.a[5] + n3 * g.a[8];
                if (sqrt(x * x + y * y + z * z) < rmax) cnt++;
            }
        }
        int total;
        int excl = block_excl_scan_256(cnt, s_warp, total);
        if (FILL && cnt > 0) {
            long long o = row_start[A] + running + excl;
            for (int n1 = lo[0]; n1 <= hi[0]; n1++) for (int n2 = lo[1]; n2 <= hi[1]; n2++) for (int n3 = lo[2]; n3 <= hi[2]; n3++) {
                double x = dx + n1 * g.a[0] + n2 * g.a[3] + n3 * g.a[6];
                double y = dy + n1 * g.a[1] + n2 * g.a[4] + n3 * g.a[7];
                double z = dz + n1 * g.a[2] + n2 * g.a[5] + n3 * g.a[8];
                if (sqrt(x * x + y * y + z * z) < rmax) { pB[o] = B; pR[3 * o] = n1; pR[3 * o + 1] = n2; pR[3 * o + 2] = n3; o++; }
            }
        }
        running += total;
    }
    if (!FILL && threadIdx.x == 0) row_count[A] = (int)running;
}

// ---------------------------------------------------------------------------------------------------
// Neighbour pass, stage A: one CTA per coarse cell (a block of cb[0] x cb[1] x cb[2] batches) lists, in image
// order, the atom images whose sphere can touch the coarse cell (fractional bounding-box test, conservative).
struct ImageDev { double x, y, z, rc; int atom, shift; };

__global__ void __launch_bounds__(256) k_coarse_candidates(Geom g, int cbx, int cby, int cbz, int ncx, int ncy, int ncz,
                                                           int n_img, const ImageDev* __restrict__ img, int cap,
                                                           int* __restrict__ cand, int* __restrict__ cand_count) {
    __shared__ int s_warp[9];
    const int cell = blockIdx.x;
    const int cz = cell % ncz, cy = (cell / ncz) % ncy, cx = cell / (ncz * ncy);
    const int cb[3] = {cbx, cby, cbz}, cc[3] = {cx, cy, cz};
    double lo[3], hi[3];
    for (int i = 0; i < 3; i++) {
        int p0 = cc[i] * cb[i] * g.bs[i];
        int p1 = min(p0 + cb[i] * g.bs[i], g.N[i]) - 1;
        lo[i] = (double)p0 / g.N[i]; hi[i] = (double)p1 / g.N[i];
    }
    int running = 0;
    for (int q0 = 0; q0 < n_img; q0 += 256) {
        const int q = q0 + threadIdx.x;
        int flag = 0;
        if (q < n_img) {
            ImageDev im = img[q];
            flag = 1;
            for (int i = 0; i < 3; i++) {
                double f = im.x * g.inv[i] + im.y * g.inv[3 + i] + im.z * g.inv[6 + i];
                double ext = im.rc / g.hgt[i] * (1.0 + 1e-12) + 1e-12;
                if (f + ext < lo[i] || f - ext > hi[i]) flag = 0;
            }
        }
        int total;
        int excl = block_excl_scan_256(flag, s_warp, total);
        if (flag && running + excl < cap) cand[(size_t)cell * cap + running + excl] = q;
        running += total;
    }
    if (threadIdx.x == 0) cand_count[cell] = running;
}

// Stage B: one warp per batch.  An image is a neighbour of the batch iff at least one batch point is closer
// than rc, decided on the same numbers the orbital evaluation uses (mesh_point()).
// COUNT pass: number of neighbours and of their orbitals.  FILL pass: the entries, sorted by falling activity
// (number of batch points inside the sphere; ties keep the (atom, shift) order) so that the atoms that are non-zero
// on every point of the batch come first and atoms with similar zero patterns share fragments of 8 orbitals;
// then the number G of atom groups the contraction kernels tile this batch with (<= GINT_TILE_ATOMS atoms and
// <= GINT_TILE_ORB orbitals per group).
template <bool FILL>
__global__ void __launch_bounds__(256) k_batch_neighbours(Geom g, int cbx, int cby, int cbz, int ncy, int ncz,
                                                          const ImageDev* __restrict__ img, int cap, const int* __restrict__ cand,
                                                          const int* __restrict__ cand_count, long long n_batch_total,
                                                          int* __restrict__ count, int* __restrict__ cols,
                                                          const SpeciesDev* __restrict__ sp, const int* __restrict__ spec,
                                                          const int* __restrict__ bstart, NeighEntry* __restrict__ bent,
                                                          int* __restrict__ bgroups) {
    __shared__ int s_act[FILL ? 8 : 1][FILL ? GINT_MAX_NB : 1];
    __shared__ int s_img[FILL ? 8 : 1][FILL ? GINT_MAX_NB : 1];
    __shared__ unsigned long long s_mlo[FILL ? 8 : 1][FILL ? GINT_MAX_NB : 1], s_mhi[FILL ? 8 : 1][FILL ? GINT_MAX_NB : 1];
    const int w = threadIdx.x >> 5;
    const long long b = (long long)blockIdx.x * 8 + w;
    const int lane = threadIdx.x & 31;
    if (b >= n_batch_total) return;
    const int bz = (int)(b % g.nb[2]), by = (int)((b / g.nb[2]) % g.nb[1]), bx = (int)(b / ((long long)g.nb[2] * g.nb[1]));
    const int i0 = bx * g.bs[0], j0 = by * g.bs[1], k0 = bz * g.bs[2];
    const int ex = min(g.bs[0], g.N[0] - i0), ey = min(g.bs[1], g.N[1] - j0), ez = min(g.bs[2], g.N[2] - k0);
    const int Kb = ex * ey * ez;
    const int cell = ((bx / cbx) * ncy + (by / cby)) * ncz + (bz / cbz);
    int n = 0, ncol = 0;
    const int nc = min(cand_count[cell], cap);
    for (int c = 0; c < nc; c++) {
        const int qi = cand[(size_t)cell * cap + c];
        const ImageDev im = img[qi];
        int hits = 0;
        unsigned mw[4] = {0u, 0u, 0u, 0u};
        for (int q = lane; q < Kb; q += 32) {
            const int qk = q % ez, qj = (q / ez) % ey, qx = q / (ez * ey);
            double px, py, pz;
            mesh_point(g, i0 + qx, j0 + qj, k0 + qk, px, py, pz);
            const double dx = px - im.x, dy = py - im.y, dz = pz - im.z;
            const bool in = fma(dx, dx, fma(dy, dy, dz * dz)) < im.rc * im.rc;    // same expression as the orbital evaluation
            hits += in;
            if (FILL && in) {
                const int cl = ((qx >> 1) * 4 + (qj >> 1)) * GINT_NCZ + qk / GINT_CZ;
#pragma unroll
                for (int wd = 0; wd < 4; wd++) if ((cl >> 5) == wd) mw[wd] |= 1u << (cl & 31);
            }
        }
#pragma unroll
        for (int d = 16; d; d >>= 1) hits += __shfl_xor_sync(0xffffffffu, hits, d);
        if (FILL) {
#pragma unroll
            for (int wd = 0; wd < 4; wd++) mw[wd] = __reduce_or_sync(0xffffffffu, mw[wd]);
        }
        if (hits > 0) {
            if (FILL && lane == 0 && n < GINT_MAX_NB) { s_act[w][n] = hits; s_img[w][n] = qi; s_mlo[w][n] = (unsigned long long)mw[0] | ((unsigned long long)mw[1] << 32); s_mhi[w][n] = (unsigned long long)mw[2] | ((unsigned long long)mw[3] << 32); }
            n++;
            ncol += sp[spec[im.atom]].norb;
        }
    }
    if (!FILL) {
        if (lane == 0) { count[b] = n; cols[b] = ncol; }
        return;
    }
    __syncwarp();
    const int base = bstart[b];
    for (int e = lane; e < n; e += 32) {                   // rank sort by (activity desc, position asc)
        const int a = s_act[w][e];
        int rank = 0;
        for (int j = 0; j < n; j++) { const int aj = s_act[w][j]; rank += (aj > a) || (aj == a && j < e); }
        const ImageDev im = img[s_img[w][e]];
        bent[base + rank].atom = im.atom; bent[base + rank].shift = im.shift;
        bent[base + rank].mask[0] = s_mlo[w][e]; bent[base + rank].mask[1] = s_mhi[w][e];
    }
    __syncwarp();
    if (lane == 0) {
        int G = (n + GINT_TILE_ATOMS - 1) / GINT_TILE_ATOMS;
        for (; G < n; G++) {
            bool ok = true;
            for (int k = 0; k < G && ok; k++) {
                int o = 0;
                for (int e = group_begin(k, n, G); e < group_begin(k + 1, n, G); e++) o += sp[spec[bent[base + e].atom]].norb;
                ok = o <= GINT_TILE_ORB;
            }
            if (ok) break;
        }
        bgroups[b] = G;
    }
}

// tile descriptors: all group pairs I <= J of every batch, batches in mesh order
__global__ void __launch_bounds__(256) k_tiles_fill(long long n_batch_total, const int* __restrict__ bgroups,
                                                    const int* __restrict__ tstart, int2* __restrict__ tile) {
    const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= n_batch_total) return;
    const int G = bgroups[b];
    int o = tstart[b];
    for (int I = 0; I < G; I++) for (int J = I; J < G; J++) tile[o++] = make_int2((int)b, I | (J << 8) | (G << 16));
}
__global__ void __launch_bounds__(256) k_tiles_count(long long n, const int* __restrict__ bgroups, int* __restrict__ tcount) {
    const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (b < n) { const int G = bgroups[b]; tcount[b] = G * (G + 1) / 2; }
}

// ---------------------------------------------------------------------------------------------------
// exclusive scan of int32 (n up to ~1e9/1024 blocks): per-block sums, scan of the sums, per-block scan + offset
__global__ void __launch_bounds__(256) k_scan_block_sums(const int* __restrict__ in, long long n, int* __restrict__ sums) {
    __shared__ int s_warp[9];
    long long base = (long long)blockIdx.x * 1024;
    int v = 0;
    for (int t = 0; t < 4; t++) { long long i = base + threadIdx.x * 4 + t; if (i < n) v += in[i]; }
    int total; block_excl_scan_256(v, s_warp, total);
    if (threadIdx.x == 0) sums[blockIdx.x] = total;
}
__global__ void __launch_bounds__(256) k_scan_apply(const int* __restrict__ in, long long n, const long long* __restrict__ block_off, int* __restrict__ out) {
    __shared__ int s_warp[9];
    long long base = (long long)blockIdx.x * 1024;
    int x[4], v = 0;
    for (int t = 0; t < 4; t++) { long long i = base + threadIdx.x * 4 + t; x[t] = i < n ? in[i] : 0; v += x[t]; }
    int total; int excl = block_excl_scan_256(v, s_warp, total);
    long long o = block_off[blockIdx.x] + excl;
    for (int t = 0; t < 4; t++) { long long i = base + threadIdx.x * 4 + t; if (i < n) out[i] = (int)o; o += x[t]; }
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 255) out[n] = (int)o;
}

// Device temporaries of the init passes: released on every way out of the scope, the early returns of GINT_CUDA / GINT_FAIL included.
template <class T> struct DevTmp {
    T* p = nullptr;
    DevTmp() = default;
    DevTmp(const DevTmp&) = delete;
    DevTmp& operator=(const DevTmp&) = delete;
    ~DevTmp() { reset(); }
    cudaError_t alloc(size_t n) { reset(); return cudaMalloc((void**)&p, sizeof(T) * (n ? n : 1)); }
    void reset() { if (p) { cudaFree(p); p = nullptr; } }
    operator T*() const { return p; }
};
struct EventTmp {
    cudaEvent_t e = nullptr;
    ~EventTmp() { if (e) cudaEventDestroy(e); }
    cudaError_t create() { return cudaEventCreate(&e); }
    operator cudaEvent_t() const { return e; }
};

// out[0..n] = exclusive scan of in[0..n); block sums are scanned on the host (n/1024 values).
int gint_device_excl_scan(const int* d_in, long long n, int* d_out, long long* total) {
    int nblk = (int)((n + 1023) / 1024);
    if (nblk == 0) { int z = 0; GINT_CUDA(cudaMemcpy(d_out, &z, sizeof(int), cudaMemcpyHostToDevice)); *total = 0; return GINT_OK; }
    DevTmp<int> d_sums; DevTmp<long long> d_off;
    GINT_CUDA(d_sums.alloc(nblk));
    GINT_CUDA(d_off.alloc(nblk));
    k_scan_block_sums<<<nblk, 256>>>(d_in, n, d_sums);
    std::vector<int> hs(nblk); std::vector<long long> ho(nblk);
    GINT_CUDA(cudaMemcpy(hs.data(), d_sums, sizeof(int) * nblk, cudaMemcpyDeviceToHost));
    long long acc = 0;
    for (int i = 0; i < nblk; i++) { ho[i] = acc; acc += hs[i]; }
    if (acc > 2000000000LL) GINT_FAIL(GINT_ERR_UNSUPPORTED, "neighbour table has %lld entries (> 2e9)", acc);
    GINT_CUDA(cudaMemcpy(d_off, ho.data(), sizeof(long long) * nblk, cudaMemcpyHostToDevice));
    k_scan_apply<<<nblk, 256>>>(d_in, n, d_off, d_out);
    GINT_CUDA(cudaGetLastError());
    GINT_CUDA(cudaDeviceSynchronize());     // the temporaries go out of scope here
    *total = acc;
    return GINT_OK;
}

// ---------------------------------------------------------------------------------------------------
// host helpers
static double det3(const double* c) {
    return c[0] * (c[4] * c[8] - c[5] * c[7]) - c[1] * (c[3] * c[8] - c[5] * c[6]) + c[2] * (c[3] * c[7] - c[4] * c[6]);
}
static void inverse3(const double* c, double* inv) {   // frac = pos * inv
    double d = det3(c);
    inv[0] = (c[4] * c[8] - c[5] * c[7]) / d; inv[1] = (c[2] * c[7] - c[1] * c[8]) / d; inv[2] = (c[1] * c[5] - c[2] * c[4]) / d;
    inv[3] = (c[5] * c[6] - c[3] * c[8]) / d; inv[4] = (c[0] * c[8] - c[2] * c[6]) / d; inv[5] = (c[2] * c[3] - c[0] * c[5]) / d;
    inv[6] = (c[3] * c[7] - c[4] * c[6]) / d; inv[7] = (c[1] * c[6] - c[0] * c[7]) / d; inv[8] = (c[0] * c[4] - c[1] * c[3]) / d;
}
static inline unsigned long long pack_key(const Geom& g, int B, int n1, int n2, int n3) {
    const unsigned long long M = (unsigned long long)g.key_M;
    return (((unsigned long long)B * M + (unsigned long long)(n1 + g.key_m)) * M + (unsigned long long)(n2 + g.key_m)) * M + (unsigned long long)(n3 + g.key_m);
}

template <class T> static int dev_alloc(gint_ctx* c, T** p, size_t n) {
    size_t bytes = sizeof(T) * (n ? n : 1);
    GINT_CUDA(cudaMalloc((void**)p, bytes));
    c->device_bytes += bytes;
    return GINT_OK;
}
template <class T> static int dev_upload(gint_ctx* c, T** p, const std::vector<T>& v) {
    int rc = dev_alloc(c, p, v.size());
    if (rc) return rc;
    if (!v.empty()) GINT_CUDA(cudaMemcpy(*p, v.data(), sizeof(T) * v.size(), cudaMemcpyHostToDevice));
    return GINT_OK;
}

static void free_ctx(gint_ctx* c) {
    if (!c) return;
    cudaFree(c->d_species); cudaFree(c->d_tab); cudaFree(c->d_atom_pos); cudaFree(c->d_atom_species);
    cudaFree(c->d_poff); cudaFree(c->d_pcanon); cudaFree(c->d_pflag); cudaFree(c->d_pnA);
    cudaFree(c->d_crow); cudaFree(c->d_ckey); cudaFree(c->d_coff); cudaFree(c->d_cpub); cudaFree(c->d_cmir); cudaFree(c->d_cval);
    cudaFree(c->d_bstart); cudaFree(c->d_bent); cudaFree(c->d_tile); cudaFree(c->d_tstart); cudaFree(c->d_gstart);
    cudaFree(c->d_goff); cudaFree(c->d_phi); cudaFree(c->d_queue); cudaFree(c->d_planoff); cudaFree(c->d_plan);
    cudaFree(c->d_stage_in); cudaFree(c->d_stage_out); cudaFree(c->d_dfull);
    for (auto& e : c->ev_force) if (e) cudaEventDestroy(e);
    for (auto& e : c->ev) if (e) cudaEventDestroy(e);
    for (auto& v : c->ev_wave) for (auto& e : v) if (e) cudaEventDestroy(e);
    for (auto& e : c->ev_copy) if (e) cudaEventDestroy(e);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    delete c;
}

// ---- step 0: basis tables -> knot-major cells {y, y'' dr^2/6} ------------------------------------------------
// R(r) = a y_i + b y_{i+1} + (a^3 - a) z_i + (b^3 - b) z_{i+1},  z = y'' dr^2/6,  b = r/dr - i, a = 1 - b   (reading R5)
// Cell (species, knot i, shell k) sits at double2 index tab_off + i * n_shell + k, so that the two knots of an
// interval are 2 * n_shell consecutive 16-byte cells.  The whole table (56 KB for the 5-shell, 701-knot basis of
// BASELINE.json) is copied into shared memory by the contraction kernels when it fits.
static int build_basis(gint_ctx* c, int n_species, const int* n_shell, const int* shell_l, const double* rcut, double dr,
                       const int* n_knot, const double* tab_y, const double* tab_y2) {
    c->n_species = n_species;
    c->h_species.resize(n_species);
    std::vector<double> tab;
    long long sh = 0, src = 0;
    int rows = 0;
    for (int s = 0; s < n_species; s++) {
        SpeciesDev& S = c->h_species[s];
        if (n_shell[s] < 1 || n_shell[s] > GINT_MAX_SHELL) GINT_FAIL(GINT_ERR_UNSUPPORTED, "species %d: %d shells (1..%d supported)", s, n_shell[s], GINT_MAX_SHELL);
        if (!(rcut[s] > 0) || !std::isfinite(rcut[s])) GINT_FAIL(GINT_ERR_INVALID_ARG, "species %d: rcut must be positive", s);
        if (n_knot[s] < 2) GINT_FAIL(GINT_ERR_INVALID_ARG, "species %d: n_knot < 2", s);
        if ((n_knot[s] - 1) * dr < rcut[s] * (1 - 1e-12)) GINT_FAIL(GINT_ERR_INVALID_ARG, "species %d: table ends at %g < rcut %g", s, (n_knot[s] - 1) * dr, rcut[s]);
        S.rc = rcut[s]; S.n_shell = n_shell[s]; S.norb = 0; S.n_int = n_knot[s] - 1; S.tab_off = rows; S.row_len = 4 * n_shell[s];
        for (int k = 0; k < n_shell[s]; k++) {
            int l = shell_l[sh + k];
            if (l < 0 || l > GINT_MAX_L) GINT_FAIL(GINT_ERR_UNSUPPORTED, "species %d shell %d: l = %d (0..%d supported)", s, k, l, GINT_MAX_L);
            S.l[k] = l; S.norb += 2 * l + 1;
        }
        if (S.norb > GINT_MAX_ORB) GINT_FAIL(GINT_ERR_UNSUPPORTED, "species %d: %d orbitals (max %d)", s, S.norb, GINT_MAX_ORB);
        S.tab_off = (int)(tab.size() / 2);
        const double h2 = dr * dr;
        for (int i = 0; i < n_knot[s]; i++) {
            for (int k = 0; k < n_shell[s]; k++) {
                const double y = tab_y[src + (long long)k * n_knot[s] + i], y2 = tab_y2[src + (long long)k * n_knot[s] + i];
                if (!std::isfinite(y) || !std::isfinite(y2))
                    GINT_FAIL(GINT_ERR_INVALID_ARG, "species %d shell %d: non-finite table value at knot %d", s, k, i);
                tab.push_back(y);
                tab.push_back(h2 / 6.0 * y2);
            }
        }
        rows += S.n_int;
        sh += n_shell[s];
        src += (long long)n_shell[s] * n_knot[s];
    }
    int rc = dev_upload(c, &c->d_species, c->h_species); if (rc) return rc;
    rc = dev_upload(c, &c->d_tab, tab); if (rc) return rc;
    c->tab_bytes = tab.size() * sizeof(double);
    return GINT_OK;
}

// ---- step a1: pair list -------------------------------------------------------------------------------
static int build_pairs(gint_ctx* c) {
    const int n = c->n_atoms;
    Geom& g = c->geom;
    DevTmp<int> d_cnt; GINT_CUDA(d_cnt.alloc(n));
    if (n > 0) k_pairs<false><<<n, 256>>>(g, n, c->d_atom_pos, c->d_atom_species, c->d_species, d_cnt, nullptr, nullptr, nullptr);
    GINT_CUDA(cudaGetLastError());
    std::vector<int> cnt(n);
    GINT_CUDA(cudaMemcpy(cnt.data(), d_cnt, sizeof(int) * n, cudaMemcpyDeviceToHost));
    std::vector<long long> rs(n + 1, 0);
    for (int i = 0; i < n; i++) rs[i + 1] = rs[i] + cnt[i];
    const long long np = rs[n];
    if (np > 2000000000LL) GINT_FAIL(GINT_ERR_UNSUPPORTED, "%lld pair keys (> 2e9)", np);
    DevTmp<long long> d_rs; DevTmp<int> d_pB, d_pR;
    GINT_CUDA(d_rs.alloc(n + 1));
    GINT_CUDA(d_pB.alloc(np));
    GINT_CUDA(d_pR.alloc(3 * np));
    GINT_CUDA(cudaMemcpy(d_rs, rs.data(), sizeof(long long) * (n + 1), cudaMemcpyHostToDevice));
    if (n > 0) k_pairs<true><<<n, 256>>>(g, n, c->d_atom_pos, c->d_atom_species, c->d_species, d_cnt, d_rs, d_pB, d_pR);
    GINT_CUDA(cudaGetLastError());
    c->n_pairs = np;
    c->h_pA.resize(np); c->h_pB.resize(np); c->h_pR.resize(3 * np); c->h_poff.resize(np + 1);
    if (np > 0) {
        GINT_CUDA(cudaMemcpy(c->h_pB.data(), d_pB, sizeof(int) * np, cudaMemcpyDeviceToHost));
        GINT_CUDA(cudaMemcpy(c->h_pR.data(), d_pR, sizeof(int) * 3 * np, cudaMemcpyDeviceToHost));
    }
    d_cnt.reset(); d_rs.reset(); d_pB.reset(); d_pR.reset();

    // host bookkeeping: offsets, canonical half, mirror map (integer work on ~1e6 keys)
    int m = 0;
    for (long long i = 0; i < 3 * np; i++) m = std::max(m, std::abs(c->h_pR[i]));
    if (m > 60) GINT_FAIL(GINT_ERR_UNSUPPORTED, "cell is too small for the cutoff: lattice shift %d > 60", m);
    g.key_m = m; g.key_M = 2 * m + 1;
    std::vector<unsigned long long> key(np);
    std::vector<int> pnab(np);
    long long off = 0;
    for (int A = 0; A < n; A++) for (long long p = rs[A]; p < rs[A + 1]; p++) {
        c->h_pA[p] = A;
        const int B = c->h_pB[p];
        const int nA = c->h_species[c->h_atom_species[A]].norb, nB = c->h_species[c->h_atom_species[B]].norb;
        c->h_poff[p] = off; off += (long long)nA * nB;
        pnab[p] = nA | (nB << 16);
        key[p] = pack_key(g, B, c->h_pR[3 * p], c->h_pR[3 * p + 1], c->h_pR[3 * p + 2]);
    }
    c->h_poff[np] = off; c->n_values = off;
    std::vector<int> pcanon(np), crow(n + 1, 0), cpub, cmir;
    std::vector<unsigned char> pflag(np);
    std::vector<unsigned long long> ckey;
    std::vector<unsigned int> coff;
    unsigned long long coffacc = 0;
    // first pass: canonical keys in list order
    for (int A = 0; A < n; A++) {
        crow[A] = (int)ckey.size();
        for (long long p = rs[A]; p < rs[A + 1]; p++) {
            const int B = c->h_pB[p]; const int* R = &c->h_pR[3 * p];
            bool ge0 = R[0] > 0 || (R[0] == 0 && (R[1] > 0 || (R[1] == 0 && R[2] >= 0)));
            bool canon = A < B || (A == B && ge0);
            pflag[p] = canon;
            if (canon) {
                pcanon[p] = (int)ckey.size();
                ckey.push_back(key[p]); cpub.push_back((int)p);
                if (coffacc > 4000000000ULL) GINT_FAIL(GINT_ERR_UNSUPPORTED, "canonical value array exceeds 2^32 doubles");
                coff.push_back((unsigned int)coffacc);
                coffacc += (unsigned long long)(pnab[p] & 0xffff) * (pnab[p] >> 16);
            }
        }
    }
    crow[n] = (int)ckey.size();
    coff.push_back((unsigned int)coffacc);
    c->n_canon = (long long)ckey.size(); c->n_cvalues = (long long)coffacc;
    cmir.resize(ckey.size());
    // second pass: mirror (B, A, -n) of every key by binary search in row B
    for (long long p = 0; p < np; p++) {
        const int A = c->h_pA[p], B = c->h_pB[p]; const int* R = &c->h_pR[3 * p];
        unsigned long long want = pack_key(g, A, -R[0], -R[1], -R[2]);
        auto b0 = key.begin() + rs[B], b1 = key.begin() + rs[B + 1];
        auto it = std::lower_bound(b0, b1, want);
        if (it == b1 || *it != want) GINT_FAIL(GINT_ERR_BAD_STATE, "internal: pair list not closed under mirroring at key %lld", p);
        long long q = it - key.begin();
        if (pflag[p]) cmir[pcanon[p]] = (int)q; else pcanon[p] = -1 - (int)q;   // resolved below
    }
    for (long long p = 0; p < np; p++) if (!pflag[p]) pcanon[p] = pcanon[-1 - pcanon[p]];
    int rc;
    if ((rc = dev_upload(c, &c->d_poff, c->h_poff))) return rc;
    if ((rc = dev_upload(c, &c->d_pcanon, pcanon))) return rc;
    if ((rc = dev_upload(c, &c->d_pflag, pflag))) return rc;
    if ((rc = dev_upload(c, &c->d_pnA, pnab))) return rc;
    if ((rc = dev_upload(c, &c->d_crow, crow))) return rc;
    if ((rc = dev_upload(c, &c->d_ckey, ckey))) return rc;
    if ((rc = dev_upload(c, &c->d_coff, coff))) return rc;
    if ((rc = dev_upload(c, &c->d_cpub, cpub))) return rc;
    if ((rc = dev_upload(c, &c->d_cmir, cmir))) return rc;
    if ((rc = dev_alloc(c, &c->d_cval, (size_t)c->n_cvalues))) return rc;
    return GINT_OK;
}

// Frees what build_batches built (the tuner builds several batch shapes in turn).
static void release_batches(gint_ctx* c) {
    cudaDeviceSynchronize();
    cudaFree(c->d_bstart); cudaFree(c->d_bent); cudaFree(c->d_tile); cudaFree(c->d_tstart); cudaFree(c->d_gstart);
    cudaFree(c->d_goff); cudaFree(c->d_phi); cudaFree(c->d_queue); cudaFree(c->d_planoff); cudaFree(c->d_plan);
    c->d_bstart = nullptr; c->d_bent = nullptr; c->d_tile = nullptr; c->d_tstart = nullptr; c->d_gstart = nullptr;
    c->d_goff = nullptr; c->d_phi = nullptr; c->d_queue = nullptr; c->d_planoff = nullptr; c->d_plan = nullptr;
    for (auto& v : c->ev_wave) { for (auto& e : v) if (e) cudaEventDestroy(e); v.clear(); }
    for (auto& e : c->ev_copy) if (e) cudaEventDestroy(e);
    c->ev_copy.clear();
    c->waves.clear();
    c->device_bytes = c->device_bytes_base;
    c->have_alg = false;
}

// ---- step a2: grid batches and their neighbour lists ------------------------------------------------------
// Tries one batch shape: fills geom.bs/nb/K/LD/max_cols/max_nb and the CSR neighbour table.  Returns
// GINT_ERR_UNSUPPORTED (without message) when the orbital tile of the largest batch does not fit in `smem_limit`.
// crop_planes > 0 (the batch-shape tuner): only the batches of the first crop_planes batch planes along a1 are built.
static int build_batches(gint_ctx* c, const int bs[3], size_t smem_limit, size_t phi_cap, bool* fits, int crop_planes = 0) {
    Geom& g = c->geom;
    *fits = false;
    for (int i = 0; i < 3; i++) { g.bs[i] = std::min(bs[i], g.N[i]); g.nb[i] = (g.N[i] + g.bs[i] - 1) / g.bs[i]; }
    if (crop_planes > 0) g.nb[0] = std::min(g.nb[0], crop_planes);
    g.K = g.bs[0] * g.bs[1] * g.bs[2];
    for (int i = 0; i < 3; i++) if (bs[i] < 1 || bs[i] > (i == 2 ? GINT_MAX_BSZ : GINT_MAX_BS)) GINT_FAIL(GINT_ERR_UNSUPPORTED, "batch edge %d (1..%d supported)", bs[i], i == 2 ? GINT_MAX_BSZ : GINT_MAX_BS);
    const long long nbt = (long long)g.nb[0] * g.nb[1] * g.nb[2];
    if (nbt > 2000000000LL) GINT_FAIL(GINT_ERR_UNSUPPORTED, "%lld batches", nbt);
    c->n_batch_total = nbt;

    // atom images whose sphere can reach the home mesh (host; O(atoms)); sorted by (atom, shift lexicographic)
    std::vector<ImageDev> img;
    for (int A = 0; A < c->n_atoms; A++) {
        const double* p = &c->h_atom_pos[3 * A];
        const double rc = c->h_species[c->h_atom_species[A]].rc;
        double f[3], ext[3]; int lo[3], hi[3];
        for (int i = 0; i < 3; i++) {
            f[i] = p[0] * g.inv[i] + p[1] * g.inv[3 + i] + p[2] * g.inv[6 + i];
            ext[i] = rc / g.hgt[i] * (1.0 + 1e-12) + 1e-12;
            lo[i] = (int)std::floor(-f[i] - ext[i]); hi[i] = (int)std::ceil(1.0 - f[i] + ext[i]);
        }
        for (int t1 = lo[0]; t1 <= hi[0]; t1++) for (int t2 = lo[1]; t2 <= hi[1]; t2++) for (int t3 = lo[2]; t3 <= hi[2]; t3++) {
            const int t[3] = {t1, t2, t3}; bool ok = true;
            for (int i = 0; i < 3; i++) {
                double fc = f[i] + t[i];
                if (fc + ext[i] < 0.0 || fc - ext[i] > (double)(g.N[i] - 1) / g.N[i]) ok = false;
            }
            if (!ok) continue;
            if (std::abs(t1) > 60 || std::abs(t2) > 60 || std::abs(t3) > 60) GINT_FAIL(GINT_ERR_UNSUPPORTED, "atom %d lies more than 60 cells away from the home cell", A);
            ImageDev im;
            image_pos(g, p, t1, t2, t3, im.x, im.y, im.z);      // the same fma chain as on the device
            im.rc = rc; im.atom = A; im.shift = pack_shift(t1, t2, t3);
            img.push_back(im);
        }
    }
    const int n_img = (int)img.size();
    DevTmp<ImageDev> d_img;
    GINT_CUDA(d_img.alloc(n_img));
    if (n_img) GINT_CUDA(cudaMemcpy(d_img, img.data(), sizeof(ImageDev) * n_img, cudaMemcpyHostToDevice));

    // stage A: coarse cells of about 16 x 16 x 8 points
    const int cb[3] = {std::max(1, 16 / g.bs[0]), std::max(1, 16 / g.bs[1]), std::max(1, 8 / g.bs[2])};
    const int nc[3] = {(g.nb[0] + cb[0] - 1) / cb[0], (g.nb[1] + cb[1] - 1) / cb[1], (g.nb[2] + cb[2] - 1) / cb[2]};
    const long long ncell = (long long)nc[0] * nc[1] * nc[2];
    int cap = 256;
    DevTmp<int> d_cand, d_ccount;
    GINT_CUDA(d_ccount.alloc(ncell));
    for (;;) {
        GINT_CUDA(d_cand.alloc((size_t)ncell * cap));
        k_coarse_candidates<<<(unsigned)ncell, 256>>>(g, cb[0], cb[1], cb[2], nc[0], nc[1], nc[2], n_img, d_img, cap, d_cand, d_ccount);
        GINT_CUDA(cudaGetLastError());
        std::vector<int> cc(ncell);
        GINT_CUDA(cudaMemcpy(cc.data(), d_ccount, sizeof(int) * ncell, cudaMemcpyDeviceToHost));
        int mx = 0; for (long long i = 0; i < ncell; i++) mx = std::max(mx, cc[i]);
        if (mx <= cap) break;
        cap = ((mx + 63) / 64) * 64;
    }
    // stage B: count, scan, fill
    DevTmp<int> d_count, d_cols;
    GINT_CUDA(d_count.alloc(nbt));
    GINT_CUDA(d_cols.alloc(nbt));
    const unsigned gridB = (unsigned)((nbt + 7) / 8);
    k_batch_neighbours<false><<<gridB, 256>>>(g, cb[0], cb[1], cb[2], nc[1], nc[2], d_img, cap, d_cand, d_ccount, nbt, d_count, d_cols,
                                              c->d_species, c->d_atom_species, nullptr, nullptr, nullptr);
    GINT_CUDA(cudaGetLastError());
    std::vector<int> count(nbt), cols(nbt);
    GINT_CUDA(cudaMemcpy(count.data(), d_count, sizeof(int) * nbt, cudaMemcpyDeviceToHost));
    GINT_CUDA(cudaMemcpy(cols.data(), d_cols, sizeof(int) * nbt, cudaMemcpyDeviceToHost));
    int max_nb = 0, max_cols = 0;
    for (long long b = 0; b < nbt; b++) { max_nb = std::max(max_nb, count[b]); max_cols = std::max(max_cols, cols[b]); }
    g.max_nb = std::max(max_nb, 1); g.max_cols = std::max(max_cols, 1);
    const bool ok = max_nb <= GINT_MAX_NB && gint_smem_needed(c, smem_limit) <= smem_limit &&     // else: try a smaller batch shape
                    (!c->want_force || gint_force_smem(c) <= smem_limit);
    if (!ok) return GINT_OK;
    *fits = true;

    int rc;
    if ((rc = dev_alloc(c, &c->d_bstart, (size_t)nbt + 1))) return rc;
    long long n_ent = 0;
    if ((rc = gint_device_excl_scan(d_count, nbt, c->d_bstart, &n_ent))) return rc;
    c->n_entries = n_ent;
    if ((rc = dev_alloc(c, &c->d_bent, (size_t)n_ent))) return rc;
    DevTmp<int> d_bgroups, d_tcount;
    GINT_CUDA(d_bgroups.alloc(nbt));
    GINT_CUDA(d_tcount.alloc(nbt));
    if ((rc = dev_alloc(c, &c->d_tstart, (size_t)nbt + 1))) return rc;
    if ((rc = dev_alloc(c, &c->d_gstart, (size_t)nbt + 1))) return rc;
    k_batch_neighbours<true><<<gridB, 256>>>(g, cb[0], cb[1], cb[2], nc[1], nc[2], d_img, cap, d_cand, d_ccount, nbt, d_count, d_cols,
                                             c->d_species, c->d_atom_species, c->d_bstart, c->d_bent, d_bgroups);
    GINT_CUDA(cudaGetLastError());
    const unsigned gridT = (unsigned)((nbt + 255) / 256);
    k_tiles_count<<<gridT, 256>>>(nbt, d_bgroups, d_tcount);
    GINT_CUDA(cudaGetLastError());
    long long n_tiles = 0, n_groups = 0;
    if ((rc = gint_device_excl_scan(d_tcount, nbt, c->d_tstart, &n_tiles))) return rc;
    if ((rc = gint_device_excl_scan(d_bgroups, nbt, c->d_gstart, &n_groups))) return rc;
    c->n_tiles = n_tiles;
    if ((rc = dev_alloc(c, &c->d_tile, (size_t)n_tiles))) return rc;
    k_tiles_fill<<<gridT, 256>>>(nbt, d_bgroups, c->d_tstart, c->d_tile);
    GINT_CUDA(cudaGetLastError());
    GINT_CUDA(cudaDeviceSynchronize());
    d_img.reset(); d_cand.reset(); d_ccount.reset(); d_count.reset(); d_cols.reset();
    d_bgroups.reset(); d_tcount.reset();
    // orbital-value ("Phi") layout: offsets of every (batch, group) slot array, waves, scratch buffer
    bool batch_too_big = false;
    if ((rc = gint_build_phi_layout(c, nullptr, phi_cap, &batch_too_big))) {
        if (!batch_too_big) return rc;
        release_batches(c);          // one batch alone overflows the scratch: this shape does not fit, a smaller one may
        *fits = false;
        return GINT_OK;
    }
    if ((rc = gint_build_plans(c))) return rc;

    c->padded_macs = 0; c->n_batch = 0;
    for (long long b = 0; b < nbt; b++) {
        if (cols[b] > 0) {
            c->n_batch++;
            int bz = (int)(b % g.nb[2]), by = (int)((b / g.nb[2]) % g.nb[1]), bx = (int)(b / ((long long)g.nb[2] * g.nb[1]));
            long long kb = (long long)std::min(g.bs[0], g.N[0] - bx * g.bs[0]) * std::min(g.bs[1], g.N[1] - by * g.bs[1]) * std::min(g.bs[2], g.N[2] - bz * g.bs[2]);
            c->padded_macs += kb * cols[b] * cols[b];
        }
    }
    c->n_batch_empty = nbt - c->n_batch;
    return GINT_OK;
}

// ---------------------------------------------------------------------------------------------------
static int gint_init_impl(gint_ctx** out, gint_ctx*& c, int n_species, const int* n_shell, const int* shell_l, const double* rcut, double dr,
                          const int* n_knot, const double* tab_y, const double* tab_y2, int n_atoms, const int* atom_species,
                          const double* atom_pos, const double cell[9], const int mesh[3], int device, unsigned long long flags) {
    if (!n_shell || !shell_l || !rcut || !n_knot || !tab_y || !tab_y2 || !cell || !mesh) GINT_FAIL(GINT_ERR_INVALID_ARG, "NULL array argument");
    if (n_species < 1) GINT_FAIL(GINT_ERR_INVALID_ARG, "n_species = %d", n_species);
    if (n_atoms < 0 || (n_atoms > 0 && (!atom_species || !atom_pos))) GINT_FAIL(GINT_ERR_INVALID_ARG, "bad atom arrays");
    if (!(dr > 0) || !std::isfinite(dr)) GINT_FAIL(GINT_ERR_INVALID_ARG, "dr must be positive");
    for (int i = 0; i < 9; i++) if (!std::isfinite(cell[i])) GINT_FAIL(GINT_ERR_INVALID_ARG, "cell has a non-finite entry");
    if (!(det3(cell) > 0)) GINT_FAIL(GINT_ERR_INVALID_ARG, "det(cell) = %g must be positive", det3(cell));
    for (int i = 0; i < 3; i++) if (mesh[i] < 1) GINT_FAIL(GINT_ERR_INVALID_ARG, "mesh[%d] = %d", i, mesh[i]);
    if ((double)mesh[0] * mesh[1] * mesh[2] > 2.0e9 * 512) GINT_FAIL(GINT_ERR_UNSUPPORTED, "mesh too large");
    for (int a = 0; a < n_atoms; a++) {
        if (atom_species[a] < 0 || atom_species[a] >= n_species) GINT_FAIL(GINT_ERR_INVALID_ARG, "atom %d: species %d out of range", a, atom_species[a]);
        for (int k = 0; k < 3; k++) if (!std::isfinite(atom_pos[3 * a + k])) GINT_FAIL(GINT_ERR_INVALID_ARG, "atom %d: non-finite position", a);
    }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1) GINT_FAIL(GINT_ERR_CUDA, "no usable CUDA device (%s); libgint has no CPU fallback", cudaGetErrorString(e));
    if (device < 0 || device >= ndev) GINT_FAIL(GINT_ERR_INVALID_ARG, "device %d of %d", device, ndev);
    GINT_CUDA(cudaSetDevice(device));
    cudaDeviceProp prop;
    GINT_CUDA(cudaGetDeviceProperties(&prop, device));
    if (prop.major < 10) GINT_FAIL(GINT_ERR_UNSUPPORTED, "device %s is sm_%d%d; libgint is built for sm_100a only", prop.name, prop.major, prop.minor);

    c = new (std::nothrow) gint_ctx();
    if (!c) GINT_FAIL(GINT_ERR_OUT_OF_MEMORY, "host allocation failed");
    c->device = device;
    Geom& g = c->geom;
    memcpy(g.a, cell, sizeof(double) * 9);
    inverse3(cell, g.inv);
    for (int i = 0; i < 3; i++) g.hgt[i] = 1.0 / std::sqrt(g.inv[i] * g.inv[i] + g.inv[3 + i] * g.inv[3 + i] + g.inv[6 + i] * g.inv[6 + i]);
    for (int i = 0; i < 3; i++) g.N[i] = mesh[i];
    g.dV = det3(cell) / ((double)mesh[0] * mesh[1] * mesh[2]);
    g.inv_dr = 1.0 / dr;
    for (int i = 0; i < 3; i++) for (int k = 0; k < 3; k++) g.step[3 * i + k] = cell[3 * i + k] / (double)mesh[i];
    c->n_atoms = n_atoms;
    c->h_atom_species.assign(atom_species, atom_species + n_atoms);
    c->h_atom_pos.assign(atom_pos, atom_pos + 3 * (size_t)n_atoms);

    int rc = build_basis(c, n_species, n_shell, shell_l, rcut, dr, n_knot, tab_y, tab_y2);
    if (rc) { return rc; }
    c->n_orb_total = 0;
    for (int a = 0; a < n_atoms; a++) c->n_orb_total += c->h_species[atom_species[a]].norb;
    if ((rc = dev_upload(c, &c->d_atom_pos, c->h_atom_pos)) || (rc = dev_upload(c, &c->d_atom_species, c->h_atom_species))) { return rc; }
    if ((rc = build_pairs(c))) { return rc; }

    const size_t smem_limit = prop.sharedMemPerBlockOptin;
    c->smem_optin = smem_limit;
    c->want_force = (flags & GINT_FLAG_FORCE) != 0;
    // scratch for the orbital values of one wave of batches: at most 16 GiB and a quarter of the free device memory, or what the caller asks for
    size_t mem_free = 0, mem_total = 0;
    GINT_CUDA(cudaMemGetInfo(&mem_free, &mem_total));
    size_t phi_cap = std::min<size_t>((size_t)16 << 30, mem_free / 4);
    if (const unsigned long long mb = (flags >> 40) & 0xfffffull) phi_cap = (size_t)mb << 20;   // GINT_FLAG_PHI_CAP_MB
    for (auto& e : c->ev) if (cudaEventCreate(&e) != cudaSuccess) { GINT_FAIL(GINT_ERR_CUDA, "cudaEventCreate failed"); }
    for (auto& e : c->ev_force) if (cudaEventCreate(&e) != cudaSuccess) { GINT_FAIL(GINT_ERR_CUDA, "cudaEventCreate failed"); }
    const int fx = (int)(flags & 255), fy = (int)((flags >> 8) & 255), fz = (int)((flags >> 16) & 255);
    c->device_bytes_base = c->device_bytes;
    bool fits = false;
    int tuned[3] = {0, 0, 0};
    if ((flags & GINT_FLAG_TUNE) && !(fx || fy || fz) && n_atoms > 0) {
        // Online tuning of the grid-batch shape (kernels of several tile sizes are tried at start-up on a task of fixed
        // size, "no more than two seconds"): every candidate shape is built for a slab of the mesh (about GINT_TUNE_BATCHES batches,
        // whole batch planes along a1), gint_vlocal + gint_rho run on it twice with V = 1, D = 1, and the shape with the least time per
        // covered mesh plane is kept.
        // The first candidate is the untuned default; another shape replaces it only if it wins by GINT_TUNE_MARGIN (the shapes
        // often lie within 1 % of each other, and the choice also fixes memory, plan size and the order of summation: it should not
        // flip from run to run on timing noise).  Each candidate's time is the least of GINT_TUNE_REPS runs after one warm-up run.
        // A candidate that cannot be built or run is recorded with -1 and skipped; if the tuning buffers themselves cannot be
        // allocated, init goes on untuned.
        static const int cand[][3] = {{8, 8, 16}, {8, 8, 8}, {4, 8, 16}, {4, 4, 16}, {4, 4, 8}};
        const auto t_begin = std::chrono::steady_clock::now();
        const size_t plane = (size_t)mesh[1] * mesh[2];
        // the same slab of the mesh for every candidate: the planes that GINT_TUNE_BATCHES batches of the largest shape cover
        const long long per_plane16 = (long long)((mesh[1] + 7) / 8) * ((mesh[2] + 15) / 16);
        const int planes16 = std::max(2, (int)((GINT_TUNE_BATCHES + per_plane16 - 1) / per_plane16));
        int crop[sizeof(cand) / sizeof(cand[0])], slab = 0;
        for (size_t k = 0; k < sizeof(cand) / sizeof(cand[0]); k++) {
            const int bs0 = std::min(cand[k][0], mesh[0]);
            crop[k] = std::max(1, planes16 * 8 / bs0);
            slab = std::max(slab, std::min(mesh[0], crop[k] * bs0));
        }
        DevTmp<double> d_V, d_rho, d_D, d_H;
        EventTmp e0, e1;
        const size_t nval = (size_t)std::max<long long>(c->n_values, 1);
        c->tune.clear();
        bool have_buffers = d_V.alloc(slab * plane) == cudaSuccess && d_rho.alloc(slab * plane) == cudaSuccess && d_D.alloc(nval) == cudaSuccess &&
                            d_H.alloc(nval) == cudaSuccess && e0.create() == cudaSuccess && e1.create() == cudaSuccess;
        if (!have_buffers) cudaGetLastError();      // out of memory for the tuner is not an error of gint_init
        if (have_buffers) {   // 1.0 everywhere (an exact zero would be skipped by the flush of gint_vlocal)
            std::vector<double> ones(1 << 20, 1.0);
            for (size_t o = 0; o < slab * plane; o += ones.size()) GINT_CUDA(cudaMemcpy(d_V + o, ones.data(), sizeof(double) * std::min(ones.size(), slab * plane - o), cudaMemcpyHostToDevice));
            for (size_t o = 0; o < (size_t)c->n_values; o += ones.size()) GINT_CUDA(cudaMemcpy(d_D + o, ones.data(), sizeof(double) * std::min(ones.size(), (size_t)c->n_values - o), cudaMemcpyHostToDevice));
        }
        for (size_t k = 0; have_buffers && k < sizeof(cand) / sizeof(cand[0]); k++) {
            const int* s = cand[k];
            gint_ctx::TuneResult tr; tr.bs[0] = s[0]; tr.bs[1] = s[1]; tr.bs[2] = s[2]; tr.ns_per_point = -1.0;
            c->rho_planes = slab;                   // gint_rho clears only the slab while tuning
            int trc = build_batches(c, s, smem_limit, phi_cap, &fits, crop[k]);
            if (trc == GINT_OK && fits && c->n_tiles > 0) {
                c->smem_bytes = gint_smem_needed(c, smem_limit);
                trc = gint_configure_kernels(c);
                float ms_best = -1.f;
                for (int rep = 0; trc == GINT_OK && rep < 1 + GINT_TUNE_REPS; rep++) {
                    cudaEventRecord(e0, 0);
                    if ((trc = gint_launch_vlocal(c, d_V, d_H, 0)) || (trc = gint_launch_rho(c, d_D, d_rho, 0))) break;
                    cudaEventRecord(e1, 0);
                    float ms = 0.f;
                    if (cudaEventSynchronize(e1) != cudaSuccess || cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) { trc = GINT_ERR_CUDA; break; }
                    if (rep > 0 && (ms_best < 0.f || ms < ms_best)) ms_best = ms;
                }
                if (trc == GINT_OK && ms_best >= 0.f)
                    tr.ns_per_point = 1e6 * ms_best / ((double)std::min(mesh[0], c->geom.nb[0] * c->geom.bs[0]) * mesh[1] * mesh[2]);
            }
            if (trc != GINT_OK) {
                // a sticky device error cannot be skipped; anything else (out of memory, unsupported shape) only drops this candidate
                cudaGetLastError();
                if (cudaDeviceSynchronize() != cudaSuccess) { c->rho_planes = 0; GINT_FAIL(GINT_ERR_CUDA, "tuner: %s", cudaGetErrorString(cudaGetLastError())); }
            }
            c->tune.push_back(tr);
            release_batches(c);
            c->timed[0] = c->timed[1] = false;
        }
        c->rho_planes = 0;
        {   // the default (first row) stays unless the fastest other shape beats it by the margin
            int kb = -1;
            for (size_t k = 1; k < c->tune.size(); k++) if (c->tune[k].ns_per_point > 0 && (kb < 0 || c->tune[k].ns_per_point < c->tune[kb].ns_per_point)) kb = (int)k;
            const double t_default = c->tune.empty() ? -1.0 : c->tune[0].ns_per_point;
            if (t_default > 0 && !(kb >= 0 && c->tune[kb].ns_per_point < t_default * (1.0 - GINT_TUNE_MARGIN))) kb = 0;
            if (kb >= 0) { tuned[0] = c->tune[kb].bs[0]; tuned[1] = c->tune[kb].bs[1]; tuned[2] = c->tune[kb].bs[2]; }
        }
        c->tune_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count();
        fits = false;
    }
    // the tuned shape was timed on a slab; should the whole mesh not fit it, the untuned ladder below takes over
    if (tuned[0] && (rc = build_batches(c, tuned, smem_limit, phi_cap, &fits))) { return rc; }
    if (fits) {
    } else if (fx || fy || fz) {
        const int bs[3] = {fx ? fx : 8, fy ? fy : 8, fz ? fz : 8};
        if ((rc = build_batches(c, bs, smem_limit, phi_cap, &fits))) { return rc; }
        if (!fits) { GINT_FAIL(GINT_ERR_UNSUPPORTED, "requested batch %dx%dx%d needs more shared memory than %zu bytes (or > %d neighbours)", bs[0], bs[1], bs[2], smem_limit, GINT_MAX_NB); }
    } else {
        static const int shapes[][3] = {{8, 8, GINT_MAX_BSZ}, {8, 8, 8}, {4, 4, 8}, {4, 4, 4}, {2, 2, 4}, {1, 1, 4}, {1, 1, 1}};
        for (auto& s : shapes) {
            if ((rc = build_batches(c, s, smem_limit, phi_cap, &fits))) { return rc; }
            if (fits) break;
        }
        if (!fits) { GINT_FAIL(GINT_ERR_UNSUPPORTED, "even a 1-point batch does not fit: too many overlapping atoms"); }
    }
    c->smem_bytes = gint_smem_needed(c, smem_limit);
    if ((rc = gint_configure_kernels(c))) { return rc; }
    if (cudaDeviceSynchronize() != cudaSuccess) { GINT_FAIL(GINT_ERR_CUDA, "gint_init: device error %s", cudaGetErrorString(cudaGetLastError())); }
    *out = c;
    return GINT_OK;
}

// The C boundary: nothing is thrown across it (std::vector of up to 2e9 keys can run out of host memory), every failure frees what
// was built so far, and the caller's current device is restored.
extern "C" int gint_init(gint_ctx** out, int n_species, const int* n_shell, const int* shell_l, const double* rcut, double dr,
                         const int* n_knot, const double* tab_y, const double* tab_y2, int n_atoms, const int* atom_species,
                         const double* atom_pos, const double cell[9], const int mesh[3], int device, unsigned long long flags) {
    if (!out) GINT_FAIL(GINT_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    DeviceGuard guard;
    gint_ctx* c = nullptr;
    int rc;
    try {
        rc = gint_init_impl(out, c, n_species, n_shell, shell_l, rcut, dr, n_knot, tab_y, tab_y2, n_atoms, atom_species, atom_pos, cell, mesh, device, flags);
    } catch (const std::bad_alloc&) {
        gint_set_error("gint_init: out of host memory");
        rc = GINT_ERR_OUT_OF_MEMORY;
    } catch (...) {
        gint_set_error("gint_init: unexpected exception");
        rc = GINT_ERR_BAD_STATE;
    }
    if (rc != GINT_OK) {
        if (c) { cudaDeviceSynchronize(); free_ctx(c); }
        *out = nullptr;
    }
    return rc;
}

extern "C" int gint_free(gint_ctx* ctx) {
    if (!ctx) GINT_FAIL(GINT_ERR_BAD_STATE, "NULL context");
    DeviceGuard guard;
    cudaSetDevice(ctx->device);
    cudaDeviceSynchronize();
    free_ctx(ctx);
    return GINT_OK;
}

extern "C" int gint_n_orb(const gint_ctx* ctx, long long* n) {
    if (!ctx) GINT_FAIL(GINT_ERR_BAD_STATE, "NULL context");
    if (!n) GINT_FAIL(GINT_ERR_INVALID_ARG, "NULL output");
    *n = ctx->n_orb_total; return GINT_OK;
}
extern "C" int gint_n_pairs(const gint_ctx* ctx, long long* n_pairs, long long* n_values) {
    if (!ctx) GINT_FAIL(GINT_ERR_BAD_STATE, "NULL context");
    if (n_pairs) *n_pairs = ctx->n_pairs;
    if (n_values) *n_values = ctx->n_values;
    return GINT_OK;
}
extern "C" int gint_get_pairs(const gint_ctx* ctx, int* A, int* B, int* R3, long long* offset) {
    if (!ctx) GINT_FAIL(GINT_ERR_BAD_STATE, "NULL context");
    const size_t n = (size_t)ctx->n_pairs;
    if (A && n) memcpy(A, ctx->h_pA.data(), sizeof(int) * n);
    if (B && n) memcpy(B, ctx->h_pB.data(), sizeof(int) * n);
    if (R3 && n) memcpy(R3, ctx->h_pR.data(), sizeof(int) * 3 * n);
    if (offset) memcpy(offset, ctx->h_poff.data(), sizeof(long long) * (n + 1));
    return GINT_OK;
}

extern "C" int gint_stats(gint_ctx* ctx, long long* out) {
    if (!ctx) GINT_FAIL(GINT_ERR_BAD_STATE, "NULL context");
    if (!out) GINT_FAIL(GINT_ERR_INVALID_ARG, "NULL output");
    DeviceGuard guard;
    if (!ctx->have_alg) { int rc = gint_launch_alg_stats(ctx); if (rc) return rc; }
    const Geom& g = ctx->geom;
    out[GINT_STAT_N_BATCH] = ctx->n_batch; out[GINT_STAT_N_BATCH_EMPTY] = ctx->n_batch_empty;
    out[GINT_STAT_BATCH_BX] = g.bs[0]; out[GINT_STAT_BATCH_BY] = g.bs[1]; out[GINT_STAT_BATCH_BZ] = g.bs[2];
    out[GINT_STAT_NEIGH_ENTRIES] = ctx->n_entries; out[GINT_STAT_MAX_NB] = g.max_nb; out[GINT_STAT_MAX_COLS] = g.max_cols;
    out[GINT_STAT_PADDED_MACS] = ctx->padded_macs; out[GINT_STAT_N_CANON] = ctx->n_canon;
    out[GINT_STAT_ALG_INCIDENCE] = ctx->alg[0]; out[GINT_STAT_ALG_SUM_N] = ctx->alg[1]; out[GINT_STAT_ALG_SUM_N2] = ctx->alg[2];
    out[GINT_STAT_NONEMPTY_POINTS] = ctx->alg[3];
    out[GINT_STAT_SMEM_BYTES] = (long long)ctx->smem_bytes; out[GINT_STAT_DEVICE_BYTES] = (long long)ctx->device_bytes;
    out[GINT_STAT_LAUNCHES_VLOCAL] = 1 + 2 * (long long)ctx->waves.size(); out[GINT_STAT_LAUNCHES_RHO] = 1 + 2 * (long long)ctx->waves.size();
    out[GINT_STAT_SMEM_EVAL] = (long long)ctx->smem_eval; out[GINT_STAT_TAB_IN_SMEM] = ctx->tab_in_smem ? 1 : 0;
    out[GINT_STAT_PHI_BYTES] = (long long)(ctx->phi_rows_total * GINT_ROW_BYTES); out[GINT_STAT_PHI_SCRATCH_BYTES] = (long long)ctx->phi_bytes;
    out[GINT_STAT_N_WAVES] = (long long)ctx->waves.size(); out[GINT_STAT_N_TILES] = ctx->n_tiles;
    out[GINT_STAT_TUNE_US] = (long long)(1e6 * ctx->tune_seconds);
    return GINT_OK;
}

extern "C" int gint_kernel_times(gint_ctx* ctx, double out[2]) {
    if (!ctx) GINT_FAIL(GINT_ERR_BAD_STATE, "NULL context");
    if (!out) GINT_FAIL(GINT_ERR_INVALID_ARG, "NULL output");
    DeviceGuard guard;
    GINT_CUDA(cudaSetDevice(ctx->device));
    for (int k = 0; k < 2; k++) {
        out[k] = -1.0;
        if (!ctx->timed[k]) continue;
        float ms = 0.f;
        GINT_CUDA(cudaEventSynchronize(ctx->ev[2 * k + 1]));
        GINT_CUDA(cudaEventElapsedTime(&ms, ctx->ev[2 * k], ctx->ev[2 * k + 1]));
        out[k] = 1e-3 * (double)ms;
    }
    return GINT_OK;
}

extern "C" int gint_phase_times(gint_ctx* ctx, double out[4]) {
    if (!ctx) GINT_FAIL(GINT_ERR_BAD_STATE, "NULL context");
    if (!out) GINT_FAIL(GINT_ERR_INVALID_ARG, "NULL output");
    DeviceGuard guard;
    GINT_CUDA(cudaSetDevice(ctx->device));
    for (int k = 0; k < 2; k++) {
        out[2 * k] = out[2 * k + 1] = -1.0;
        if (!ctx->timed[k] || ctx->ev_wave[k].empty()) continue;
        double te = 0.0, tt = 0.0;
        cudaEvent_t prev = ctx->ev[2 * k];
        for (size_t w = 0; w < ctx->ev_wave[k].size(); w++) {
            float ms = 0.f;
            GINT_CUDA(cudaEventSynchronize(ctx->ev_wave[k][w]));
            GINT_CUDA(cudaEventElapsedTime(&ms, prev, ctx->ev_wave[k][w]));
            ((w & 1) ? tt : te) += 1e-3 * (double)ms;
            prev = ctx->ev_wave[k][w];
        }
        out[2 * k] = te; out[2 * k + 1] = tt;
    }
    return GINT_OK;
}

// ---- host-buffer entry points (end-to-end path) ------------------------------------------------------------
static int ensure_stage(gint_ctx* c, double** p, size_t* have, size_t want) {
    if (*have >= want) return GINT_OK;
    if (*p) { cudaFree(*p); c->device_bytes -= *have * sizeof(double); *p = nullptr; *have = 0; }
    GINT_CUDA(cudaMalloc((void**)p, sizeof(double) * want));
    *have = want; c->device_bytes += want * sizeof(double);
    return GINT_OK;
}
extern "C" int gint_vlocal_host(gint_ctx* c, const double* V_host, double* H_host, void* stream) {
    if (!c) GINT_FAIL(GINT_ERR_BAD_STATE, "NULL context");
    if (!V_host || !H_host) GINT_FAIL(GINT_ERR_INVALID_ARG, "NULL buffer");
    DeviceGuard guard;
    cudaStream_t st = (cudaStream_t)stream;
    GINT_CUDA(cudaSetDevice(c->device));
    const size_t npts = (size_t)c->geom.N[0] * c->geom.N[1] * c->geom.N[2];
    int rc;
    if ((rc = ensure_stage(c, &c->d_stage_in, &c->stage_in_n, std::max(npts, (size_t)c->n_values)))) return rc;
    if ((rc = ensure_stage(c, &c->d_stage_out, &c->stage_out_n, std::max(npts, (size_t)c->n_values)))) return rc;
    // V goes up in chunks on the copy stream, ahead of the waves that read it
    if ((rc = gint_launch_vlocal(c, c->d_stage_in, c->d_stage_out, st, V_host))) return rc;
    GINT_CUDA(cudaMemcpyAsync(H_host, c->d_stage_out, sizeof(double) * (size_t)c->n_values, cudaMemcpyDeviceToHost, st));
    GINT_CUDA(cudaStreamSynchronize(st));
    return GINT_OK;
}
extern "C" int gint_rho_host(gint_ctx* c, const double* D_host, double* rho_host, void* stream) {
    if (!c) GINT_FAIL(GINT_ERR_BAD_STATE, "NULL context");
    if (!D_host || !rho_host) GINT_FAIL(GINT_ERR_INVALID_ARG, "NULL buffer");
    DeviceGuard guard;
    cudaStream_t st = (cudaStream_t)stream;
    GINT_CUDA(cudaSetDevice(c->device));
    const size_t npts = (size_t)c->geom.N[0] * c->geom.N[1] * c->geom.N[2];
    int rc;
    if ((rc = ensure_stage(c, &c->d_stage_in, &c->stage_in_n, std::max(npts, (size_t)c->n_values)))) return rc;
    if ((rc = ensure_stage(c, &c->d_stage_out, &c->stage_out_n, std::max(npts, (size_t)c->n_values)))) return rc;
    GINT_CUDA(cudaMemcpyAsync(c->d_stage_in, D_host, sizeof(double) * (size_t)c->n_values, cudaMemcpyHostToDevice, st));
    // rho comes down in chunks on the copy stream, each behind the wave that completes it
    if ((rc = gint_launch_rho(c, c->d_stage_in, c->d_stage_out, st, rho_host))) return rc;
    GINT_CUDA(cudaStreamSynchronize(st));
    return GINT_OK;
}
extern "C" int gint_vlocal(gint_ctx* c, const double* V_dev, double* H_dev, void* stream) {
    if (!c) GINT_FAIL(GINT_ERR_BAD_STATE, "NULL context");
    if (!V_dev || (!H_dev && c->n_values)) GINT_FAIL(GINT_ERR_INVALID_ARG, "NULL device pointer");
    if (((uintptr_t)V_dev | (uintptr_t)H_dev) & 7) GINT_FAIL(GINT_ERR_INVALID_ARG, "device pointers must be 8-byte aligned");
    DeviceGuard guard;
    return gint_launch_vlocal(c, V_dev, H_dev, (cudaStream_t)stream);
}
extern "C" int gint_rho(gint_ctx* c, const double* D_dev, double* rho_dev, void* stream) {
    if (!c) GINT_FAIL(GINT_ERR_BAD_STATE, "NULL context");
    if ((!D_dev && c->n_values) || !rho_dev) GINT_FAIL(GINT_ERR_INVALID_ARG, "NULL device pointer");
    if (((uintptr_t)D_dev | (uintptr_t)rho_dev) & 7) GINT_FAIL(GINT_ERR_INVALID_ARG, "device pointers must be 8-byte aligned");
    DeviceGuard guard;
    return gint_launch_rho(c, D_dev, rho_dev, (cudaStream_t)stream);
}

// ---- Pulay force and stress (Eq. 4, Eq. 5) ------------------------------------------------------------------
extern "C" int gint_force_stress(gint_ctx* c, const double* V_dev, const double* D_dev, double* F_dev, double* sigma_dev, void* stream) {
    if (!c) GINT_FAIL(GINT_ERR_BAD_STATE, "NULL context");
    if (!V_dev || (!D_dev && c->n_values) || (!F_dev && c->n_atoms)) GINT_FAIL(GINT_ERR_INVALID_ARG, "NULL device pointer");
    if (((uintptr_t)V_dev | (uintptr_t)D_dev | (uintptr_t)F_dev | (uintptr_t)sigma_dev) & 7) GINT_FAIL(GINT_ERR_INVALID_ARG, "device pointers must be 8-byte aligned");
    DeviceGuard guard;
    return gint_launch_force(c, V_dev, D_dev, F_dev, sigma_dev, (cudaStream_t)stream);
}
extern "C" int gint_force_time(gint_ctx* ctx, double* seconds) {
    if (!ctx) GINT_FAIL(GINT_ERR_BAD_STATE, "NULL context");
    if (!seconds) GINT_FAIL(GINT_ERR_INVALID_ARG, "NULL output");
    DeviceGuard guard;
    GINT_CUDA(cudaSetDevice(ctx->device));
    *seconds = -1.0;
    if (ctx->timed_force) {
        GINT_CUDA(cudaEventSynchronize(ctx->ev_force[1]));
        float ms = 0.f;
        GINT_CUDA(cudaEventElapsedTime(&ms, ctx->ev_force[0], ctx->ev_force[1]));
        *seconds = 1e-3 * ms;
    }
    return GINT_OK;
}

extern "C" int gint_tune_report(const gint_ctx* ctx, int max_rows, double* out, int* n_rows) {
    if (!ctx) GINT_FAIL(GINT_ERR_BAD_STATE, "NULL context");
    if (!out || !n_rows || max_rows < 0) GINT_FAIL(GINT_ERR_INVALID_ARG, "bad output arguments");
    int n = 0;
    for (const auto& t : ctx->tune) {
        if (n >= max_rows) break;
        out[4 * n] = t.bs[0]; out[4 * n + 1] = t.bs[1]; out[4 * n + 2] = t.bs[2]; out[4 * n + 3] = t.ns_per_point;
        n++;
    }
    *n_rows = n;
    return GINT_OK;
}
