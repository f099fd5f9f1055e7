"""Seeded synthetic workloads (inputs only) for the grid-integration path.

This module serves BOTH the CPU oracle (oracle/) and the CUDA path.  It holds none of
the method's arithmetic: no orbital evaluation, no pair enumeration, no mesh integration.
It only produces *input data*: cell, mesh, atoms, tabulated radial functions (values and
spline second derivatives, which the API takes as data), the local potential V on the mesh,
and density-matrix blocks D for a pair list supplied by the caller.

Recipe = BASELINE.json configs[0..4] with the readings of DESIGN.md "Input recipe"
(SURVEY.md section 8c A7, A11-A16).  These structures STAND IN FOR the paper's twisted
bilayer graphene structure files, which are external.
"""
from __future__ import annotations

import itertools
from dataclasses import dataclass, field

import numpy as np

SEED = (2409, 9399)

# 13-orbital basis: shells s1 s2 p1 p2 d  -> (l, alpha)   (BASELINE.json configs[0])
SHELLS = ((0, 0.60), (0, 0.20), (1, 0.50), (1, 0.18), (2, 0.40))
DR = 0.01


@dataclass
class Basis:
    n_species: int
    n_shell: np.ndarray      # int32 [n_species]
    shell_l: np.ndarray      # int32 [sum n_shell]
    rcut: np.ndarray         # f64   [n_species]
    dr: float
    n_knot: np.ndarray       # int32 [n_species]
    tab_y: np.ndarray        # f64 concatenated [species][shell][knot]
    tab_y2: np.ndarray       # f64 same shape: spline second derivatives
    norm: list = field(default_factory=list)   # normalisation constants (diagnostic)

    @property
    def norb(self):
        out, k = [], 0
        for s in range(self.n_species):
            out.append(int(sum(2 * int(l) + 1 for l in self.shell_l[k:k + self.n_shell[s]])))
            k += int(self.n_shell[s])
        return out


@dataclass
class Workload:
    name: str
    cfg: int
    cell: np.ndarray          # f64 [3,3] rows a1,a2,a3 (bohr)
    mesh: np.ndarray          # int32 [3]
    atom_species: np.ndarray  # int32 [n_atoms]
    atom_pos: np.ndarray      # f64 [n_atoms,3]
    basis: Basis

    @property
    def n_atoms(self):
        return len(self.atom_species)

    @property
    def n_points(self):
        return int(np.prod(self.mesh.astype(np.int64)))


# ----------------------------------------------------------------------------- radial tables
def _spline_second_derivatives(y: np.ndarray, h: float, d0: float, dn: float) -> np.ndarray:
    """Second derivatives of the clamped cubic spline through (i*h, y_i) with end slopes d0, dn.

    Standard tridiagonal system (Thomas algorithm).  This is input-data preparation: the
    library and the oracle both receive y'' as an array.
    """
    n = len(y) - 1
    a = np.full(n + 1, h / 6.0)   # sub-diagonal
    b = np.full(n + 1, 2.0 * h / 3.0)
    c = np.full(n + 1, h / 6.0)   # super-diagonal
    rhs = np.empty(n + 1)
    rhs[1:n] = (y[2:] - 2.0 * y[1:n] + y[:n - 1]) / h
    b[0] = h / 3.0
    rhs[0] = (y[1] - y[0]) / h - d0
    b[n] = h / 3.0
    rhs[n] = dn - (y[n] - y[n - 1]) / h
    # Thomas
    cp = np.empty(n + 1)
    dp = np.empty(n + 1)
    cp[0] = c[0] / b[0]
    dp[0] = rhs[0] / b[0]
    for i in range(1, n + 1):
        m = b[i] - a[i] * cp[i - 1]
        cp[i] = c[i] / m
        dp[i] = (rhs[i] - a[i] * dp[i - 1]) / m
    y2 = np.empty(n + 1)
    y2[n] = dp[n]
    for i in range(n - 1, -1, -1):
        y2[i] = dp[i] - cp[i] * y2[i + 1]
    return y2


def radial_raw(r, l, alpha, rc):
    """R_raw(r) = r^l exp(-alpha r^2) (1-(r/rc)^2)^3 for r<rc, else 0 (BASELINE.json configs[0])."""
    r = np.asarray(r, dtype=np.float64)
    return np.where(r < rc, r ** l * np.exp(-alpha * r * r) * (1.0 - (r / rc) ** 2) ** 3, 0.0)


def make_basis(rc: float, shells=SHELLS, dr: float = DR) -> Basis:
    """One species; every shell normalised by composite Simpson on the knots, tabulated at dr."""
    n = int(round(rc / dr))
    assert abs(n * dr - rc) < 1e-9 and n % 2 == 0
    r = np.arange(n + 1) * dr
    r[-1] = rc
    ys, y2s, norms = [], [], []
    for l, alpha in shells:
        raw = radial_raw(r, l, alpha, rc)
        raw[-1] = 0.0
        f = raw * raw * r * r
        integral = dr / 3.0 * (f[0] + f[-1] + 4.0 * f[1:-1:2].sum() + 2.0 * f[2:-1:2].sum())
        N = 1.0 / np.sqrt(integral)
        y = N * raw
        d0 = N if l == 1 else 0.0         # R'(0) = N delta_{l,1};  R'(rc) = 0
        ys.append(y)
        y2s.append(_spline_second_derivatives(y, dr, d0, 0.0))
        norms.append(float(N))
    return Basis(
        n_species=1,
        n_shell=np.array([len(shells)], dtype=np.int32),
        shell_l=np.array([l for l, _ in shells], dtype=np.int32),
        rcut=np.array([rc], dtype=np.float64),
        dr=dr,
        n_knot=np.array([n + 1], dtype=np.int32),
        tab_y=np.concatenate(ys),
        tab_y2=np.concatenate(y2s),
        norm=norms,
    )


def make_gaussian_s_basis(exponents, rc: float, dr: float = DR) -> Basis:
    """Test basis: one species per exponent, one s shell R(r) = (2a/pi)^(3/4) exp(-a r^2) / Y00.

    Used by the closed-form overlap pin; rc is chosen so wide that exp(-a rc^2) < 1e-16.
    """
    n = int(round(rc / dr))
    r = np.arange(n + 1) * dr
    ys, y2s = [], []
    y00 = 0.5 / np.sqrt(np.pi)
    for a in exponents:
        y = (2.0 * a / np.pi) ** 0.75 * np.exp(-a * r * r) / y00
        ys.append(y)
        y2s.append(_spline_second_derivatives(y, dr, 0.0, float(-2 * a * rc * y[-1])))
    ns = len(exponents)
    return Basis(ns, np.ones(ns, np.int32), np.zeros(ns, np.int32), np.full(ns, rc), dr,
                 np.full(ns, n + 1, np.int32), np.concatenate(ys), np.concatenate(y2s))


# ----------------------------------------------------------------------------- structures
def diamond(ncell: int, a: float = 6.74):
    fcc = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]], dtype=np.float64)
    basis = np.vstack([fcc, fcc + 0.25])
    cells = np.array(list(itertools.product(range(ncell), repeat=3)), dtype=np.float64)
    pos = (cells[:, None, :] + basis[None, :, :]).reshape(-1, 3) * a
    return np.eye(3) * a * ncell, pos


def graphene(n: int, a: float = 4.65, c: float = 20.0):
    a1 = a * np.array([1.0, 0.0, 0.0])
    a2 = a * np.array([0.5, np.sqrt(3.0) / 2.0, 0.0])
    b = [np.zeros(3), (a1 + a2) / 3.0]
    pos = [i * a1 + j * a2 + bb + np.array([0, 0, c / 2.0]) for i in range(n) for j in range(n) for bb in b]
    return np.array([n * a1, n * a2, [0.0, 0.0, c]]), np.array(pos)


def twisted_bilayer(i: int, a: float = 4.65, d: float = 6.33, c: float = 25.0, labels: bool = False):
    """Commensurate TBG, N = 4(3i^2+3i+1) atoms, cos(theta) = (3i^2+3i+1/2)/(3i^2+3i+1).

    Layer lattice a1 = a(1,0), a2 = a(1/2, sqrt3/2), basis {0, (a1+a2)/3}; supercell
    T1 = i a1 + (i+1) a2, T2 = -(i+1) a1 + (2i+1) a2; layer 2 is layer 1 rotated about the
    origin by the angle that carries (i+1) a1 + i a2 onto T1; sites with fractional
    coordinates in [0,1)^2 are kept.  Layers at z = c/2 -/+ d/2.
    """
    a1 = a * np.array([1.0, 0.0])
    a2 = a * np.array([0.5, np.sqrt(3.0) / 2.0])
    T1 = i * a1 + (i + 1) * a2
    T2 = -(i + 1) * a1 + (2 * i + 1) * a2
    T1p = (i + 1) * a1 + i * a2
    th = np.arctan2(T1[1], T1[0]) - np.arctan2(T1p[1], T1p[0])
    Rm = np.array([[np.cos(th), -np.sin(th)], [np.sin(th), np.cos(th)]])
    Minv = np.linalg.inv(np.array([T1, T2]))
    rng = np.arange(-3 * i - 3, 3 * i + 4)
    P, Q = np.meshgrid(rng, rng, indexing="ij")
    base = P.reshape(-1, 1) * a1 + Q.reshape(-1, 1) * a2
    pts = np.vstack([base, base + (a1 + a2) / 3.0])
    sub = np.r_[np.zeros(len(base), np.int32), np.ones(len(base), np.int32)]      # sublattice of every site
    out, lab = [], []
    for layer, (R, z) in enumerate(((np.eye(2), c / 2.0 - d / 2.0), (Rm, c / 2.0 + d / 2.0))):
        Pr = pts @ R.T
        f = np.round(Pr @ Minv, 9)
        keep = np.all((f >= -1e-9) & (f < 1 - 1e-9), axis=1)
        Pk = Pr[keep]
        order = np.lexsort((Pk[:, 1], Pk[:, 0]))       # deterministic atom order
        Pk = Pk[order]
        out.append(np.c_[Pk, np.full(len(Pk), z)])
        lab.append(2 * layer + sub[keep][order])
    cell = np.array([[T1[0], T1[1], 0.0], [T2[0], T2[1], 0.0], [0.0, 0.0, c]])
    pos = np.vstack(out)
    assert len(pos) == 4 * (3 * i * i + 3 * i + 1)
    if labels:
        return cell, pos, np.concatenate(lab)          # 2 * layer + sublattice
    return cell, pos


def _mesh_for(cell, h=0.2):
    return np.array([int(round(np.linalg.norm(cell[k]) / h)) for k in range(3)], dtype=np.int32)


def concat_bases(parts) -> Basis:
    """One Basis of several species from one-species bases (tables concatenated in species order)."""
    return Basis(len(parts), np.array([len(b.shell_l) for b in parts], np.int32), np.concatenate([b.shell_l for b in parts]),
                 np.array([float(b.rcut[0]) for b in parts]), DR, np.concatenate([b.n_knot for b in parts]),
                 np.concatenate([b.tab_y for b in parts]), np.concatenate([b.tab_y2 for b in parts]),
                 norm=sum((list(b.norm) for b in parts), []))


def make_workload(cfg: int) -> Workload:
    """The five BASELINE.json configs (0..4), and 5: a MIXED-SPECIES bilayer ("m, n = orbitals per atom 1...30",
    PAPER.md:165): the geometry of cfg3 with layer 1 of species 0 (2s2p1d, 13 orbitals, rc 7) and layer 2 of two species by
    sublattice, species 1 (2s2p, 8 orbitals, rc 8) and species 2 (2s2p2d, 18 orbitals, rc 6) -- three radial tables of different
    lengths, orbital rows that do not line up with the 8-row fragments, cutoff spheres of three sizes."""
    if cfg == 5:
        cell, pos, lab = twisted_bilayer(9, labels=True)
        species = np.where(lab < 2, 0, lab - 1).astype(np.int32)
        basis = concat_bases([make_basis(7.0),
                              make_basis(8.0, shells=((0, 0.45), (0, 0.15), (1, 0.40), (1, 0.14))),
                              make_basis(6.0, shells=((0, 0.75), (0, 0.28), (1, 0.60), (1, 0.22), (2, 0.50), (2, 0.25)))])
        return Workload("cfg5 mixed-species bilayer i=9 (1084 atoms, 13/8/18 orbitals)", 5, np.ascontiguousarray(cell, np.float64),
                        _mesh_for(cell), species, np.ascontiguousarray(pos, np.float64), basis)
    if cfg == 0:
        cell, pos = diamond(1)
        mesh, rc, name = np.array([24, 24, 24], np.int32), 5.0, "cfg0 diamond-8"
    elif cfg == 1:
        cell, pos = graphene(6)
        mesh, rc, name = _mesh_for(cell), 7.0, "cfg1 graphene 6x6 (72 atoms)"
    elif cfg == 2:
        cell, pos = diamond(4)
        mesh, rc, name = _mesh_for(cell), 7.0, "cfg2 diamond 4x4x4 (512 atoms)"
    elif cfg == 3:
        cell, pos = twisted_bilayer(9)
        mesh, rc, name = _mesh_for(cell), 7.0, "cfg3 TBG i=9 (1084 atoms)"
    elif cfg == 4:
        cell, pos = twisted_bilayer(29)
        mesh, rc, name = _mesh_for(cell), 7.0, "cfg4 TBG i=29 (10444 atoms)"
    else:
        raise ValueError(cfg)
    return Workload(name, cfg, np.ascontiguousarray(cell, np.float64), mesh,
                    np.zeros(len(pos), np.int32), np.ascontiguousarray(pos, np.float64), make_basis(rc))


# ----------------------------------------------------------------------------- V on the mesh
def make_potential(w: Workload, width: float = 1.5, amp: float = -2.0, noise: float = 0.05,
                   reach: float = 8.0) -> np.ndarray:
    """V_g = sum_{A,t} amp * exp(-|r_g - tau_A - R_t|^2 / width) + noise * u_g,  u_g ~ U(-1,1).

    Requires a3 perpendicular to a1 and a2 (true for all five configs), so each Gaussian
    factorises into an in-plane and a z factor; images are included when the in-plane offset
    and the z offset are each within `reach` bohr (dropped terms < 2e-19).  Noise is drawn
    i.i.d. in mesh order g = (i*N2 + j)*N3 + k from default_rng([2409, 9399, cfg, 0]).
    """
    cell, (N1, N2, N3) = w.cell, (int(m) for m in w.mesh)
    assert abs(cell[2] @ cell[0]) < 1e-9 and abs(cell[2] @ cell[1]) < 1e-9 and abs(cell[2, 0]) + abs(cell[2, 1]) < 1e-12
    c = cell[2, 2]
    P = cell[:2, :2]                       # in-plane lattice rows
    Pinv = np.linalg.inv(P)
    h2 = 1.0 / np.linalg.norm(Pinv, axis=0)   # in-plane heights
    zmesh = np.arange(N3) * (c / N3)
    V = np.zeros((N1, N2, N3))
    zkeys = np.round(w.atom_pos[:, 2], 9)
    for z0 in np.unique(zkeys):
        sel = np.nonzero(zkeys == z0)[0]
        # 1-D z profile with periodic images
        gz = np.zeros(N3)
        for t in range(-int(np.ceil(reach / c)) - 1, int(np.ceil(reach / c)) + 2):
            dz = zmesh - z0 - t * c
            gz += np.where(np.abs(dz) < reach, np.exp(-dz * dz / width), 0.0)
        # 2-D in-plane field
        G = np.zeros((N1, N2))
        ri = np.array([reach / h2[0] * N1, reach / h2[1] * N2])
        for A in sel:
            f = w.atom_pos[A, :2] @ Pinv
            lo = np.floor(f * [N1, N2] - ri).astype(int) - 1
            hi = np.ceil(f * [N1, N2] + ri).astype(int) + 1
            ii = np.arange(lo[0], hi[0] + 1)
            jj = np.arange(lo[1], hi[1] + 1)
            x = (ii[:, None] / N1) * P[0, 0] + (jj[None, :] / N2) * P[1, 0] - w.atom_pos[A, 0]
            y = (ii[:, None] / N1) * P[0, 1] + (jj[None, :] / N2) * P[1, 1] - w.atom_pos[A, 1]
            d2 = x * x + y * y
            patch = np.where(d2 < reach * reach, np.exp(-d2 / width), 0.0)
            iw, jw = np.mod(ii, N1), np.mod(jj, N2)
            if len(ii) <= N1 and len(jj) <= N2:
                G[np.ix_(iw, jw)] += patch
            else:
                np.add.at(G, (iw[:, None], jw[None, :]), patch)
        V += amp * G[:, :, None] * gz[None, None, :]
    rng = np.random.default_rng([*SEED, w.cfg, 0])
    V += noise * (2.0 * rng.random(N1 * N2 * N3) - 1.0).reshape(N1, N2, N3)
    return np.ascontiguousarray(V.reshape(-1))


# ----------------------------------------------------------------------------- D blocks
def mirror_index(pA, pB, pR) -> np.ndarray:
    """Index of the key (B, A, -R) for every key (A, B, R) of a complete pair list."""
    pA = np.asarray(pA, np.int64); pB = np.asarray(pB, np.int64); pR = np.asarray(pR, np.int64).reshape(-1, 3)
    n = int(max(pA.max(), pB.max())) + 1
    m = int(np.abs(pR).max()) if len(pR) else 0
    M = 2 * m + 1

    def pack(a, b, r):
        return (((a * n + b) * M + (r[:, 0] + m)) * M + (r[:, 1] + m)) * M + (r[:, 2] + m)
    keys = pack(pA, pB, pR)
    order = np.argsort(keys, kind="stable")
    want = pack(pB, pA, -pR)
    pos = np.searchsorted(keys[order], want)
    assert np.all(pos < len(keys)) and np.all(keys[order][pos] == want), "pair list is not closed under mirroring"
    return order[pos]


def make_density_blocks(w: Workload, pA, pB, pR, offset, scale_len2: float = 20.0) -> np.ndarray:
    """D values for a caller-supplied pair list (A, B, R, offset): canonical keys (A<B, or A==B and
    R >= 0 lexicographically) get a random symmetric block with N(0,1) entries times
    exp(-d^2/scale_len2), d = |tau_B + R - tau_A|; the mirror key gets the transpose.
    Drawn in pair-list order from default_rng([2409, 9399, cfg, 1]).  Uniform norb only.
    """
    pA = np.asarray(pA); pB = np.asarray(pB); pR = np.asarray(pR).reshape(-1, 3)
    offset = np.asarray(offset, np.int64)
    norb = w.basis.norb
    if len(set(norb)) != 1:
        return _make_density_blocks_mixed(w, pA, pB, pR, offset, scale_len2)
    no = norb[0]
    npairs = len(pA)
    assert offset[-1] == npairs * no * no
    r0, r1, r2 = pR[:, 0], pR[:, 1], pR[:, 2]
    lex_ge0 = (r0 > 0) | ((r0 == 0) & ((r1 > 0) | ((r1 == 0) & (r2 >= 0))))
    canon = (pA < pB) | ((pA == pB) & lex_ge0)
    mir = mirror_index(pA, pB, pR)
    d = np.linalg.norm(w.atom_pos[pB] + pR @ w.cell - w.atom_pos[pA], axis=1)
    rng = np.random.default_rng([*SEED, w.cfg, 1])
    idx = np.nonzero(canon)[0]
    D = np.zeros((npairs, no, no))
    chunk = 65536
    for s in range(0, len(idx), chunk):
        q = idx[s:s + chunk]
        g = rng.standard_normal((len(q), no, no))
        g = np.triu(g) + np.transpose(np.triu(g, 1), (0, 2, 1))
        g *= np.exp(-d[q] ** 2 / scale_len2)[:, None, None]
        D[q] = g
        selfm = mir[q] == q
        D[mir[q][~selfm]] = np.transpose(g[~selfm], (0, 2, 1))
    return np.ascontiguousarray(D.reshape(-1))


def _make_density_blocks_mixed(w: Workload, pA, pB, pR, offset, scale_len2: float) -> np.ndarray:
    """The same recipe for species with different orbital counts: the canonical key (A, B, R) gets N(0,1) entries times
    exp(-d^2/scale_len2) (symmetrised when it is its own mirror), the mirror key the transpose; one block at a time."""
    no = np.asarray(w.basis.norb)[w.atom_species]
    r0, r1, r2 = pR[:, 0], pR[:, 1], pR[:, 2]
    lex_ge0 = (r0 > 0) | ((r0 == 0) & ((r1 > 0) | ((r1 == 0) & (r2 >= 0))))
    canon = (pA < pB) | ((pA == pB) & lex_ge0)
    mir = mirror_index(pA, pB, pR)
    d = np.linalg.norm(w.atom_pos[pB] + pR @ w.cell - w.atom_pos[pA], axis=1)
    rng = np.random.default_rng([*SEED, w.cfg, 1])
    D = np.zeros(int(offset[-1]))
    for q in np.nonzero(canon)[0]:
        nA, nB = int(no[pA[q]]), int(no[pB[q]])
        g = rng.standard_normal((nA, nB)) * np.exp(-d[q] ** 2 / scale_len2)
        if mir[q] == q:
            g = np.triu(g) + np.triu(g, 1).T
        D[offset[q]:offset[q + 1]] = g.ravel()
        if mir[q] != q:
            D[offset[mir[q]]:offset[mir[q] + 1]] = g.T.ravel()
    return D
