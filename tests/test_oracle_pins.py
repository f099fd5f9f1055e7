"""Pins of the CPU oracle (oracle/gint_oracle.c) against what the paper and the mathematics fix.

None of these tests calls the CUDA path.  Each pin is independent of the oracle's own code:
  P1  H_(A,B,n) = H_(B,A,-n)^T                        (Eq. 2, PAPER.md:66 is symmetric in mu,nu)
  P2  V == 1  =>  H = S; the on-site block equals delta_ll' delta_mm' * int R_s R_s' r^2 dr
      (orthonormality of spherical harmonics; radial integrals by scipy.integrate.quad of the
      ANALYTIC radial functions of BASELINE.json configs[0], not of the tables)
  P3  sum_g rho_g dV = sum_p <D_p, S_p>               (Eq. 3, PAPER.md:73 integrated)
  P4  sum_g V_g rho_g dV = sum_p <D_p, H_p>           (Eq. 2 and Eq. 3 contracted with each other)
  P5  two normalised s Gaussians: S = (2 sqrt(ab)/(a+b))^(3/2) exp(-ab d^2/(a+b))   (textbook closed form)
  P6  brute force on 2 atoms in a skew cell with self-images: numpy loops over every mesh point x every
      image in a fixed +-3 shell, radial part by scipy.interpolate.CubicSpline (clamped), angular part
      from scipy.special.sph_harm_y -- no lists, no lens boxes, no code shared with the oracle
  P6b the same brute force on a skew 3-atom cell with TWO species that differ in rc, in the number of knots
      and in their shell sets (s,p,d / s,s,p): pins the per-species table offsets and shell look-ups
  P7  invariances: translation by one mesh step, atom permutation, linearity in V and D
  P9  pair counts against a KD-tree count; lexicographic key order
  Y   real spherical harmonics: orthonormal under Gauss-Legendre x uniform-phi quadrature
  S   spline: reproduces knots; second-derivative data from the generator equals scipy's clamped spline
"""
import itertools

import numpy as np
import pytest
from scipy.integrate import quad
from scipy.interpolate import CubicSpline
from scipy.spatial import cKDTree
from scipy.special import sph_harm_y

from oracle import oracle as O
from paper_2409_09399_b200 import workloads as W


# ----------------------------------------------------------------------------- helpers (independent of oracle/)
def real_ylm_scipy(l, ux, uy, uz):
    """Real (tesseral) harmonics m=-l..l built from scipy's complex Y_l^m (Condon-Shortley included there)."""
    theta = np.arccos(np.clip(uz, -1.0, 1.0))
    phi = np.arctan2(uy, ux)
    out = []
    for m in range(-l, l + 1):
        if m == 0:
            out.append(sph_harm_y(l, 0, theta, phi).real)
        elif m > 0:
            out.append(np.sqrt(2.0) * (-1) ** m * sph_harm_y(l, m, theta, phi).real)
        else:
            out.append(np.sqrt(2.0) * (-1) ** m * sph_harm_y(l, -m, theta, phi).imag)
    return out


def brute_phi(basis, species, d):
    """phi_{s,m}(d) for an array of displacement vectors d[...,3]; scipy spline + scipy harmonics."""
    d = np.asarray(d, np.float64)
    r = np.sqrt((d * d).sum(-1))
    rc = basis.rcut[species]
    nk = int(basis.n_knot[species])
    sh0 = int(np.sum(basis.n_shell[:species]))
    tab0 = int(sum(int(basis.n_knot[s]) * int(basis.n_shell[s]) for s in range(species)))
    knots = np.arange(nk) * basis.dr
    inside = r < rc
    rs = np.where(r > 1e-12, r, 1.0)
    ux, uy, uz = d[..., 0] / rs, d[..., 1] / rs, d[..., 2] / rs
    cols = []
    for s in range(int(basis.n_shell[species])):
        l = int(basis.shell_l[sh0 + s])
        y = basis.tab_y[tab0 + s * nk: tab0 + (s + 1) * nk]
        # end slopes of the analytic functions: R'(0) = N delta_{l,1} (y[1]/dr to O(dr^2) for l=1), R'(rc) = 0
        d0 = basis.norm[sh0 + s] if (l == 1 and basis.norm) else 0.0
        cs = CubicSpline(knots, y, bc_type=((1, d0), (1, 0.0)))
        R = np.where(inside, cs(np.minimum(r, rc)), 0.0)
        for ylm in real_ylm_scipy(l, ux, uy, uz):
            v = R * ylm
            if l > 0:
                v = np.where(r > 1e-12, v, 0.0)
            cols.append(v)
    return np.stack(cols, -1)


def mesh_points(w):
    N1, N2, N3 = (int(x) for x in w.mesh)
    i, j, k = np.meshgrid(np.arange(N1), np.arange(N2), np.arange(N3), indexing="ij")
    f = np.stack([i.ravel() / N1, j.ravel() / N2, k.ravel() / N3], -1)
    return f @ w.cell


def dV(w):
    return abs(np.linalg.det(w.cell)) / w.n_points


def small_skew_workload(rc=3.0, seed=5):
    basis = W.make_basis(rc)
    cell = np.array([[5.2, 0.0, 0.0], [1.1, 5.6, 0.0], [0.4, -0.7, 6.1]])
    pos = np.array([[0.31, 0.47, 0.59], [2.9, 3.3, 3.7]])
    return W.Workload("skew-2", 90 + seed, cell, np.array([13, 14, 15], np.int32), np.zeros(2, np.int32), pos, basis)


def brute_pairs(w, S=3):
    rc = w.basis.rcut
    keys = []
    for A in range(w.n_atoms):
        for B in range(w.n_atoms):
            for n in itertools.product(range(-S, S + 1), repeat=3):
                dvec = w.atom_pos[B] + np.array(n) @ w.cell - w.atom_pos[A]
                if np.linalg.norm(dvec) < rc[w.atom_species[A]] + rc[w.atom_species[B]]:
                    keys.append((A, B) + n)
    return sorted(keys)


# ----------------------------------------------------------------------------- fixtures
@pytest.fixture(scope="module")
def cfg0():
    w = W.make_workload(0)
    pl = O.pairs(w)
    V = W.make_potential(w)
    D = W.make_density_blocks(w, *pl)
    H = O.vlocal(w, V, pl)
    rho = O.rho(w, D, pl)
    S = O.vlocal(w, np.ones(w.n_points), pl)
    return dict(w=w, pl=pl, V=V, D=D, H=H, rho=rho, S=S)


# ----------------------------------------------------------------------------- Y: harmonics
def test_real_harmonics_orthonormal_and_match_scipy():
    basis = W.make_basis(5.0)
    x, wq = np.polynomial.legendre.leggauss(12)
    nphi = 16
    phis = (np.arange(nphi) + 0.3) * 2 * np.pi / nphi
    r0 = 1.234
    G = np.zeros((13, 13))
    Rs = None
    for ct, wt in zip(x, wq):
        st = np.sqrt(1 - ct * ct)
        for ph in phis:
            u = np.array([st * np.cos(ph), st * np.sin(ph), ct])
            v = O.phi(basis, 0, r0 * u)
            ref = brute_phi(basis, 0, r0 * u)
            assert np.allclose(v, ref, rtol=0, atol=1e-12)
            if Rs is None:
                # radial factors at r0 from the l=0 / p_z / d_z2 components
                Rs = True
            G += np.outer(v, v) * wt * 2 * np.pi / nphi
    # G[mu,nu] = R_s(r0) R_s'(r0) delta_ll' delta_mm'  -> off-diagonal (different l or m) vanish
    R = np.array([O.phi(basis, 0, np.array([0, 0, r0]))[i] for i in (0, 1)]) / 0.28209479177387814
    for a in range(13):
        for b in range(13):
            la = 0 if a < 2 else (1 if a < 8 else 2)
            lb = 0 if b < 2 else (1 if b < 8 else 2)
            ma = 0 if a < 2 else ((a - 2) % 3 if a < 8 else a - 8)
            mb = 0 if b < 2 else ((b - 2) % 3 if b < 8 else b - 8)
            if la != lb or ma != mb:
                assert abs(G[a, b]) < 1e-13, (a, b, G[a, b])
    assert abs(G[0, 0] - R[0] ** 2) < 1e-13 and abs(G[0, 1] - R[0] * R[1]) < 1e-13
    # every m of one shell has the same norm (R_s^2)
    assert np.allclose(np.diag(G)[2:5], G[2, 2], atol=1e-13) and np.allclose(np.diag(G)[8:13], G[8, 8], atol=1e-13)


def test_phi_cutoff_and_origin():
    basis = W.make_basis(5.0)
    assert np.all(O.phi(basis, 0, np.array([5.0, 0, 0])) == 0.0)          # |d| = rc is OUTSIDE (strict <)
    assert np.all(O.phi(basis, 0, np.array([3.0, 4.0, 1e-9])) == 0.0)
    inside = O.phi(basis, 0, np.array([3.0, 3.9, 0.0]))
    assert np.any(inside != 0.0)
    v0 = O.phi(basis, 0, np.zeros(3))
    assert np.allclose(v0[:2], np.array(basis.norm[:2]) * 0.28209479177387814, rtol=1e-14) and np.all(v0[2:] == 0.0)


# ----------------------------------------------------------------------------- S: spline data
SURVEY_P8_NORMS = {5.0: (1.98381907454532, 1.10072344658646, 1.62880549788493, 0.690466095447584, 0.863637740254984),
                   7.0: (1.85514473075244, 0.931663800594847, 1.4235833205831, 0.505992851061471, 0.681962212656393)}


@pytest.mark.parametrize("rc", [5.0, 7.0])
def test_spline_tables(rc):
    basis = W.make_basis(rc)
    nk = int(basis.n_knot[0])
    knots = np.arange(nk) * basis.dr
    rng = np.random.default_rng(1)
    rr = rng.uniform(0, rc, 200)
    for s, (l, alpha) in enumerate(W.SHELLS):
        y = basis.tab_y[s * nk:(s + 1) * nk]
        y2 = basis.tab_y2[s * nk:(s + 1) * nk]
        d0 = basis.norm[s] if l == 1 else 0.0
        cs = CubicSpline(knots, y, bc_type=((1, d0), (1, 0.0)))
        assert np.allclose(cs(knots, 2), y2, rtol=0, atol=1e-7 * max(1.0, np.abs(y2).max()))
        # normalisation: int R^2 r^2 dr = 1 by adaptive quadrature of the ANALYTIC function
        I, _ = quad(lambda r: W.radial_raw(r, l, alpha, rc) ** 2 * r * r, 0, rc, epsabs=1e-15, epsrel=1e-13)
        assert abs(basis.norm[s] - 1 / np.sqrt(I)) < 1e-12 * basis.norm[s]
        # SURVEY.md section 8(c) pin P8 prints these constants (bar 1e-13)
        assert abs(basis.norm[s] - SURVEY_P8_NORMS[rc][s]) <= 1e-13 * basis.norm[s]
        # oracle's interpolation vs the analytic function (interpolation error of a dr=0.01 clamped spline)
        if l == 0:
            vals = np.array([O.phi(basis, 0, np.array([0, 0, r]))[s] for r in rr]) / 0.28209479177387814
            exact = basis.norm[s] * W.radial_raw(rr, l, alpha, rc)
            assert np.abs(vals - exact).max() < 2e-9


# ----------------------------------------------------------------------------- P1..P4 on cfg0
def test_P1_H_symmetry(cfg0):
    A, B, R, off = cfg0["pl"]
    mir = W.mirror_index(A, B, R)
    H = cfg0["H"].reshape(-1, 13, 13)
    err = np.abs(H - np.transpose(H[mir], (0, 2, 1))).max()
    assert err <= 1e-13 * np.abs(H).max()
    assert np.abs(H).max() > 0.1


def _radial_overlap(i, j, rc):
    l, a1 = W.SHELLS[i]
    _, a2 = W.SHELLS[j]
    f = lambda r, a, b: W.radial_raw(r, l, a, rc) * W.radial_raw(r, l, b, rc) * r * r
    n1, _ = quad(f, 0, rc, args=(a1, a1), epsabs=1e-15, epsrel=1e-13)
    n2, _ = quad(f, 0, rc, args=(a2, a2), epsabs=1e-15, epsrel=1e-13)
    I, _ = quad(f, 0, rc, args=(a1, a2), epsabs=1e-15, epsrel=1e-13)
    return I / np.sqrt(n1 * n2)


def test_P2_overlap_onsite_closed_form(cfg0):
    """V == 1 gives S; S_(A,A,0) = delta_ll' delta_mm' int R_s R_s' r^2 dr (values also in SURVEY.md P2)."""
    A, B, R, off = cfg0["pl"]
    S = cfg0["S"].reshape(-1, 13, 13)
    E = np.eye(13)
    E[0, 1] = E[1, 0] = _radial_overlap(0, 1, 5.0)
    for m in range(3):
        E[2 + m, 5 + m] = E[5 + m, 2 + m] = _radial_overlap(2, 3, 5.0)
    assert abs(E[0, 1] - 0.896242205888) < 1e-11 and abs(E[2, 5] - 0.872169641102) < 1e-11
    onsite = np.nonzero((A == B) & np.all(R == 0, axis=1))[0]
    assert len(onsite) == 8
    for p in onsite:
        assert np.abs(S[p] - E).max() < 1e-8, np.abs(S[p] - E).max()


def test_P3_charge_equals_trace_DS(cfg0):
    w = cfg0["w"]
    q = cfg0["rho"].sum() * dV(w)
    t = float(cfg0["D"] @ cfg0["S"])
    assert abs(q - t) <= 1e-12 * max(abs(t), np.abs(cfg0["D"] * cfg0["S"]).sum())


def test_P4_V_rho_equals_D_H(cfg0):
    w = cfg0["w"]
    lhs = float(cfg0["V"] @ cfg0["rho"]) * dV(w)
    rhs = float(cfg0["D"] @ cfg0["H"])
    assert abs(lhs - rhs) <= 1e-12 * np.abs(cfg0["D"] * cfg0["H"]).sum()


# ----------------------------------------------------------------------------- P5 Gaussian closed form
@pytest.mark.parametrize("a,b,d", [(0.5, 0.3, 1.5), (0.5, 0.5, 0.0), (0.3, 0.3, 2.25)])
def test_P5_gaussian_overlap_closed_form(a, b, d):
    rc = 9.0
    basis = W.make_gaussian_s_basis([a, b], rc)
    L = 22.0
    n = 80                                     # h = 0.275 bohr
    cell = np.eye(3) * L
    pos = np.array([[L / 2 + 0.013, L / 2 - 0.021, L / 2 - d / 2 + 0.007], [L / 2 + 0.013, L / 2 - 0.021, L / 2 + d / 2 + 0.007]])
    w = W.Workload("gauss", 99, cell, np.array([n, n, n], np.int32), np.array([0, 1], np.int32), pos, basis)
    pA, pB, pR, off = O.pairs(w)
    sel = np.nonzero((pA == 0) & (pB == 1) & np.all(pR == 0, axis=1))[0]
    assert len(sel) == 1
    S = O.vlocal(w, np.ones(w.n_points), (pA, pB, pR, off), sel=sel)
    got = S[off[sel[0]]]
    want = (2 * np.sqrt(a * b) / (a + b)) ** 1.5 * np.exp(-a * b * d * d / (a + b))
    if (a, b, d) == (0.5, 0.3, 1.5):
        assert abs(want - 0.6248279851709736) < 1e-15
    assert abs(got - want) < 5e-9, (got, want)


# ----------------------------------------------------------------------------- P6 brute force
@pytest.fixture(scope="module")
def skew():
    w = small_skew_workload()
    S_ = 3
    pts = mesh_points(w)
    shell = list(itertools.product(range(-S_, S_ + 1), repeat=3))
    Phi = {}
    for A in range(w.n_atoms):
        for t in shell:
            v = brute_phi(w.basis, 0, pts - w.atom_pos[A] - np.array(t) @ w.cell)
            if np.any(v != 0.0):
                Phi[(A, t)] = v
    rng = np.random.default_rng(11)
    V = rng.normal(size=w.n_points)
    keys = brute_pairs(w, S_)
    return dict(w=w, Phi=Phi, V=V, keys=keys, shell=shell)


def test_P9_pair_list_is_brute_force_list(skew):
    A, B, R, off = O.pairs(skew["w"])
    got = [(int(a), int(b), int(r[0]), int(r[1]), int(r[2])) for a, b, r in zip(A, B, R)]
    assert got == skew["keys"]
    assert np.all(np.diff(off) == 169) and off[0] == 0
    assert any(a == b and (n1, n2, n3) != (0, 0, 0) for a, b, n1, n2, n3 in got)   # self-image keys are exercised


def test_P6_brute_force_H(skew):
    w, Phi, V = skew["w"], skew["Phi"], skew["V"]
    pl = O.pairs(w)
    H = O.vlocal(w, V, pl).reshape(-1, 13, 13)
    scale = np.abs(H).max()
    for p, (A, B, n1, n2, n3) in enumerate(skew["keys"]):
        ref = np.zeros((13, 13))
        for (A2, t), pa in Phi.items():
            if A2 != A:
                continue
            pb = Phi.get((B, (t[0] + n1, t[1] + n2, t[2] + n3)))
            if pb is not None:
                ref += pa.T @ (V[:, None] * pb)
        ref *= dV(w)
        assert np.abs(H[p] - ref).max() <= 1e-12 * scale, (p, np.abs(H[p] - ref).max())


def test_P6_brute_force_rho(skew):
    w, Phi = skew["w"], skew["Phi"]
    pl = O.pairs(w)
    rng = np.random.default_rng(12)
    D = rng.normal(size=int(pl[3][-1]))                       # NOT symmetric: every ordered block independent
    rho = O.rho(w, D, pl)
    Db = D.reshape(-1, 13, 13)
    ref = np.zeros(w.n_points)
    for p, (A, B, n1, n2, n3) in enumerate(skew["keys"]):
        for (A2, t), pa in Phi.items():
            if A2 != A:
                continue
            pb = Phi.get((B, (t[0] + n1, t[1] + n2, t[2] + n3)))
            if pb is not None:
                ref += ((pa @ Db[p]) * pb).sum(1)
    assert np.abs(rho - ref).max() <= 1e-12 * np.abs(ref).max()
    # selected-outputs mode returns the same numbers
    sel = np.array([0, 7, 1234, w.n_points - 1], np.int64)
    part = O.rho(w, D, pl, sel=sel)
    assert np.array_equal(part[sel], rho[sel]) and np.count_nonzero(part) <= len(sel)


# ----------------------------------------------------------------------------- P6b brute force, two species
def two_species_workload():
    """Skew cell, 3 atoms, species 0 = (s,p,d) with rc 3.0 (301 knots), species 1 = (s,s,p) with rc 2.5 (251 knots):
    different cutoffs, table lengths, shell sets and orbital counts (9 / 5); atoms outside the home cell; self images."""
    b0 = W.make_basis(3.0, shells=((0, 0.7), (1, 0.5), (2, 0.45)))
    b1 = W.make_basis(2.5, shells=((0, 0.9), (0, 0.3), (1, 0.6)))
    basis = W.Basis(2, np.array([3, 3], np.int32), np.concatenate([b0.shell_l, b1.shell_l]), np.array([3.0, 2.5]), W.DR,
                    np.concatenate([b0.n_knot, b1.n_knot]), np.concatenate([b0.tab_y, b1.tab_y]),
                    np.concatenate([b0.tab_y2, b1.tab_y2]), norm=b0.norm + b1.norm)
    cell = np.array([[4.9, 0.2, 0.0], [1.3, 4.4, 0.1], [0.3, -0.6, 5.1]])
    pos = np.array([[0.2, 0.4, 0.5], [2.6, 2.9, 3.1], [6.3, -0.8, 4.0]])
    return W.Workload("skew-3-two-species", 96, cell, np.array([12, 11, 13], np.int32), np.array([0, 1, 1], np.int32), pos, basis)


@pytest.fixture(scope="module")
def skew2():
    w = two_species_workload()
    S_ = 3
    pts = mesh_points(w)
    Phi = {}
    for A in range(w.n_atoms):
        for t in itertools.product(range(-S_, S_ + 1), repeat=3):
            v = brute_phi(w.basis, int(w.atom_species[A]), pts - w.atom_pos[A] - np.array(t) @ w.cell)
            if np.any(v != 0.0):
                Phi[(A, t)] = v
    return dict(w=w, Phi=Phi, keys=brute_pairs(w, S_))


def test_P6b_two_species_phi_and_pairs(skew2):
    w = skew2["w"]
    assert w.basis.norb == [9, 5] and list(w.basis.n_knot) == [301, 251]
    rng = np.random.default_rng(31)
    for sp in (0, 1):
        for _ in range(40):
            d = rng.normal(size=3) * 1.2
            assert np.allclose(O.phi(w.basis, sp, d), brute_phi(w.basis, sp, d), rtol=0, atol=1e-12)
    A, B, R, off = O.pairs(w)
    got = [(int(a), int(b), int(r[0]), int(r[1]), int(r[2])) for a, b, r in zip(A, B, R)]
    assert got == skew2["keys"]
    no = np.array(w.basis.norb)[w.atom_species]
    assert np.array_equal(np.diff(off), no[A] * no[B])
    assert {(int(a), int(b)) for a, b in zip(w.atom_species[A], w.atom_species[B])} == {(0, 0), (0, 1), (1, 0), (1, 1)}


def test_P6b_two_species_brute_force_H_and_rho(skew2):
    w, Phi, keys = skew2["w"], skew2["Phi"], skew2["keys"]
    pl = O.pairs(w)
    off = pl[3]
    no = np.array(w.basis.norb)[w.atom_species]
    rng = np.random.default_rng(32)
    V = rng.normal(size=w.n_points)
    D = rng.normal(size=int(off[-1]))                        # every ordered block independent
    H = O.vlocal(w, V, pl)
    rho = O.rho(w, D, pl)
    Href = np.zeros_like(H)
    rref = np.zeros(w.n_points)
    for p, (A, B, n1, n2, n3) in enumerate(keys):
        blk = np.zeros((no[A], no[B]))
        Dp = D[off[p]:off[p + 1]].reshape(no[A], no[B])
        for (A2, t), pa in Phi.items():
            if A2 != A:
                continue
            pb = Phi.get((B, (t[0] + n1, t[1] + n2, t[2] + n3)))
            if pb is not None:
                blk += pa.T @ (V[:, None] * pb)
                rref += ((pa @ Dp) * pb).sum(1)
        Href[off[p]:off[p + 1]] = (blk * dV(w)).ravel()
    assert np.abs(H - Href).max() <= 1e-12 * np.abs(Href).max()
    assert np.abs(rho - rref).max() <= 1e-12 * np.abs(rref).max()


# ----------------------------------------------------------------------------- P7 invariances
def test_P7_translation_by_mesh_step(skew):
    w, V = skew["w"], skew["V"]
    pl = O.pairs(w)
    rng = np.random.default_rng(13)
    D = rng.normal(size=int(pl[3][-1]))
    H0 = O.vlocal(w, V, pl)
    r0 = O.rho(w, D, pl)
    N = [int(x) for x in w.mesh]
    step = w.cell[0] / N[0] * 2 + w.cell[2] / N[2] * 5       # 2 steps along a1, 5 along a3
    w2 = W.Workload(w.name, w.cfg, w.cell, w.mesh, w.atom_species, w.atom_pos + step, w.basis)
    V2 = np.roll(V.reshape(N), (2, 5), axis=(0, 2)).reshape(-1)
    pl2 = O.pairs(w2)
    assert all(np.array_equal(x, y) for x, y in zip(pl, pl2))
    H1 = O.vlocal(w2, V2, pl2)
    r1 = O.rho(w2, D, pl2)
    assert np.abs(H1 - H0).max() <= 1e-12 * np.abs(H0).max()
    assert np.abs(np.roll(r0.reshape(N), (2, 5), axis=(0, 2)).reshape(-1) - r1).max() <= 1e-12 * np.abs(r0).max()


def test_P7_permutation_and_linearity(skew):
    w, V = skew["w"], skew["V"]
    pl = O.pairs(w)
    A, B, R, off = pl
    rng = np.random.default_rng(14)
    V2 = rng.normal(size=w.n_points)
    H_a, H_b = O.vlocal(w, V, pl), O.vlocal(w, V2, pl)
    H_ab = O.vlocal(w, 0.7 * V - 1.3 * V2, pl)
    assert np.abs(H_ab - (0.7 * H_a - 1.3 * H_b)).max() <= 1e-12 * np.abs(H_a).max()
    D1, D2 = rng.normal(size=int(off[-1])), rng.normal(size=int(off[-1]))
    assert np.abs(O.rho(w, 2 * D1 + D2, pl) - (2 * O.rho(w, D1, pl) + O.rho(w, D2, pl))).max() <= 1e-11
    # swap the two atoms: block (A,B,n) of the new system is block (1-A,1-B,n) of the old one
    w2 = W.Workload(w.name, w.cfg, w.cell, w.mesh, w.atom_species, w.atom_pos[::-1].copy(), w.basis)
    pl2 = O.pairs(w2)
    H2 = O.vlocal(w2, V, pl2).reshape(-1, 169)
    old = {(int(a), int(b), *map(int, r)): i for i, (a, b, r) in enumerate(zip(A, B, R))}
    Hb = H_a.reshape(-1, 169)
    for i, (a, b, r) in enumerate(zip(*pl2[:3])):
        j = old[(1 - int(a), 1 - int(b), *map(int, r))]
        assert np.abs(H2[i] - Hb[j]).max() <= 1e-12 * np.abs(Hb).max()


# ----------------------------------------------------------------------------- P9 structure counts
@pytest.mark.parametrize("cfg,natoms,npairs", [(0, 8, 984), (1, 72, 4824), (2, 512, 150016), (3, 1084, 129372)])
def test_P9_pair_counts_vs_kdtree(cfg, natoms, npairs):
    w = W.make_workload(cfg)
    assert w.n_atoms == natoms
    A, B, R, off = O.pairs(w)
    assert len(A) == npairs
    rc2 = 2 * w.basis.rcut[0]
    m = [int(np.ceil(rc2 / h)) for h in 1.0 / np.linalg.norm(np.linalg.inv(w.cell), axis=0)]
    shifts = np.array(list(itertools.product(*[range(-k, k + 1) for k in m]))) @ w.cell
    allpos = (w.atom_pos[None, :, :] + shifts[:, None, :]).reshape(-1, 3)
    tree = cKDTree(allpos)
    cnt = sum(len(x) for x in tree.query_ball_point(w.atom_pos, rc2 * (1 - 1e-13)))
    assert cnt == npairs
    key = np.c_[A, B, R].astype(np.int64)
    assert np.all(np.diff(np.ravel_multi_index((key + [0, 0, 8, 8, 8]).T, (natoms, natoms, 17, 17, 17))) > 0)


def test_table2_tbg_family():
    """PAPER.md:203-210 Table 2: atom counts and in-plane cell lengths of the TBG family (fixture, Angstrom)."""
    import os
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "paper_table2.txt")) if l.strip() and l[0] != "#"]
    bohr = 1.8897259886
    for row, i in zip(rows, (2, 6, 12, 29)):
        n = int(row[0])
        X = np.array(row[1:4], float)
        Z = np.array(row[7:10], float)
        assert n == 4 * (3 * i * i + 3 * i + 1)
        # garbled-column reading: in-plane vectors are X and Z (60 degrees, equal length)
        assert abs(np.linalg.norm(X) - np.linalg.norm(Z)) < 2e-2
        cell, pos = W.twisted_bilayer(i)                        # all four cells of the table, i = 29 (10,444 atoms) included
        assert len(pos) == n
        assert abs(np.linalg.norm(cell[0]) / bohr - np.linalg.norm(X)) < 2e-3 * np.linalg.norm(X)
        assert abs(np.dot(cell[0], cell[1]) / np.linalg.norm(cell[0]) ** 2 - 0.5) < 1e-12
    w4 = W.make_workload(4)
    assert w4.n_atoms == 10444 and tuple(w4.mesh) == (1188, 1188, 125)
    assert abs(np.linalg.norm(w4.cell[0]) / bohr - np.linalg.norm(np.array(rows[3][1:4], float))) < 2e-3 * 125.7
    d = cKDTree(w4.atom_pos).query(w4.atom_pos, k=2)[0][:, 1]
    assert abs(d.min() - 4.65 / np.sqrt(3)) < 1e-9            # no overlapping atoms: shortest bond = a/sqrt(3)


def test_P9_cfg4_pair_count_by_kdtree():
    """SURVEY.md P9 at the headline size: 1,246,278 ordered pair keys (|tau_B + n.cell - tau_A| < 2 rc, strict; reading R7), counted
    here with a KD-tree over the periodic images, independent of oracle_pairs (which takes minutes at this size and is compared key
    by key with this count, and with the library's list, in the GPU test of cfg4)."""
    w = W.make_workload(4)
    rc2 = 2 * w.basis.rcut[0]
    m = [int(np.ceil(rc2 / h)) for h in 1.0 / np.linalg.norm(np.linalg.inv(w.cell), axis=0)]
    shifts = np.array(list(itertools.product(*[range(-k, k + 1) for k in m]))) @ w.cell
    allpos = (w.atom_pos[None, :, :] + shifts[:, None, :]).reshape(-1, 3)
    cnt = sum(len(x) for x in cKDTree(allpos).query_ball_point(w.atom_pos, rc2 * (1 - 1e-13)))
    assert cnt == 1246278


# ----------------------------------------------------------------------------- P10 Pulay force and stress (Eq. 4, Eq. 5; reading R15)
def _energy(w, V, D, pl):
    """E = <D, H> (= dV sum_g V_g rho_g, identity P4) through the oracle's H."""
    return float(D @ O.vlocal(w, V, pl))


def test_P10_orbital_gradient_is_the_derivative_of_phi(skew2):
    """oracle_dphi against central differences (Richardson, O(h^4)) of oracle_phi and of the scipy-based brute_phi."""
    w = skew2["w"]
    rng = np.random.default_rng(41)
    h = 2e-3
    for sp in (0, 1):
        for _ in range(25):
            d = rng.normal(size=3) * 1.1
            val, grad = O.dphi(w.basis, sp, d)
            assert np.array_equal(val, O.phi(w.basis, sp, d))
            for a in range(3):
                e = np.zeros(3); e[a] = 1.0
                for f in (lambda x: O.phi(w.basis, sp, x), lambda x: brute_phi(w.basis, sp, x)):
                    fd = (8.0 * (f(d + 0.5 * h * e) - f(d - 0.5 * h * e)) - (f(d + h * e) - f(d - h * e))) / (6.0 * h)
                    assert np.abs(grad[:, a] - fd).max() <= 2e-8 * max(1.0, np.abs(grad).max()), (sp, d, a)
    # outside the sphere everything vanishes; at the nucleus only the p orbitals have a gradient (c_1 R'(0) e_m, m = y, z, x)
    val, grad = O.dphi(w.basis, 0, np.array([0.0, 0.0, 3.0]))
    assert not val.any() and not grad.any()
    val, grad = O.dphi(w.basis, 0, np.zeros(3))
    assert not grad[0].any() and not grad[4:].any()
    p = grad[1:4]                                       # rows: p_y, p_z, p_x
    assert abs(p[0, 1]) > 0.1 and p[0, 1] == p[1, 2] == p[2, 0] and np.count_nonzero(p) == 3
    eps = 1e-6
    assert abs(O.phi(w.basis, 0, np.array([0.0, eps, 0.0]))[1] / eps - p[0, 1]) <= 1e-6 * abs(p[0, 1])


def test_P10_force_is_minus_dE_dtau(cfg0):
    """F_C = -dE/dtau_C at fixed V, D, by central differences of E = <D, H> through oracle_vlocal (which P1..P9 pin)."""
    w, pl, V, D = cfg0["w"], cfg0["pl"], cfg0["V"], cfg0["D"]
    rng = np.random.default_rng(42)
    D = D + 0.3 * rng.standard_normal(D.size)           # no symmetry of D assumed
    F, sigma = O.force_stress(w, V, D, pl)
    Fsel, none = O.force_stress(w, V, D, pl, sel=np.array([5, 2]))
    assert none is None and np.array_equal(Fsel[[2, 5]], F[[2, 5]]) and not Fsel[[0, 1, 3, 4, 6, 7]].any()
    scale = np.abs(F).max()
    assert scale > 1e-3
    h = 1e-4
    for C, a in ((0, 0), (3, 1), (6, 2), (5, 0)):
        Ep = []
        for sgn in (+1, -1):
            pos = w.atom_pos.copy(); pos[C, a] += sgn * h
            Ep.append(_energy(W.Workload(w.name, w.cfg, w.cell, w.mesh, w.atom_species, pos, w.basis), V, D, pl))
        fd = -(Ep[0] - Ep[1]) / (2 * h)
        assert abs(F[C, a] - fd) <= 1e-6 * scale, (C, a, F[C, a], fd)


def test_P10_stress_is_minus_dE_deps_over_volume(skew2):
    """sigma^{ab} = -(1/Omega) dE/d eps_ab at fixed V (per mesh index), D and dV, under r -> (1 + eps) r of atoms and mesh points.
    The oracle's E carries dV = det(cell) / N, which the strain also changes: that part, delta_ab E, is taken out."""
    w = skew2["w"]
    pl = O.pairs(w)
    rng = np.random.default_rng(43)
    V = rng.normal(size=w.n_points); D = rng.normal(size=int(pl[3][-1]))
    F, sigma = O.force_stress(w, V, D, pl)
    Omega = abs(np.linalg.det(w.cell))
    E0 = _energy(w, V, D, pl)
    h = 1e-5
    for a in range(3):
        for b in range(3):
            Ep = []
            for sgn in (+1, -1):
                S = np.eye(3); S[a, b] += sgn * h              # r'_a = r_a + eps_ab r_b  (row vectors: r' = r S^T)
                ws = W.Workload(w.name, w.cfg, w.cell @ S.T, w.mesh, w.atom_species, w.atom_pos @ S.T, w.basis)
                Ep.append(_energy(ws, V, D, pl))
            dE = (Ep[0] - Ep[1]) / (2 * h) - (E0 if a == b else 0.0)
            assert abs(sigma[a, b] + dE / Omega) <= 2e-6 * np.abs(sigma).max(), (a, b, sigma[a, b], -dE / Omega)


def test_P10_brute_force_force_and_stress(skew2):
    """Independent restatement on the skew two-species cell: scipy splines and harmonics, orbital gradients by Richardson
    differences of brute_phi, plain loops over keys, images and mesh points."""
    w, Phi, keys = skew2["w"], skew2["Phi"], skew2["keys"]
    pl = O.pairs(w)
    off = pl[3]
    no = np.array(w.basis.norb)[w.atom_species]
    rng = np.random.default_rng(44)
    V = rng.normal(size=w.n_points); D = rng.normal(size=int(off[-1]))
    F, sigma = O.force_stress(w, V, D, pl)
    index = {k: p for p, k in enumerate(keys)}
    pts = mesh_points(w)
    h = 2e-3
    Fref = np.zeros((w.n_atoms, 3)); sref = np.zeros((3, 3))
    Omega = abs(np.linalg.det(w.cell))
    for (C, t), pc in Phi.items():
        sp = int(w.atom_species[C])
        d = pts - w.atom_pos[C] - np.array(t) @ w.cell
        psi = np.zeros((w.n_points, no[C]))
        for (C2, B, n1, n2, n3), p in index.items():
            if C2 != C:
                continue
            pb = Phi.get((B, (t[0] + n1, t[1] + n2, t[2] + n3)))
            if pb is None:
                continue
            q = index[(B, C, -n1, -n2, -n3)]
            Dsym = D[off[p]:off[p + 1]].reshape(no[C], no[B]) + D[off[q]:off[q + 1]].reshape(no[B], no[C]).T
            psi += pb @ Dsym.T
        for a in range(3):
            e = np.zeros(3); e[a] = 1.0
            g = (8.0 * (brute_phi(w.basis, sp, d + 0.5 * h * e) - brute_phi(w.basis, sp, d - 0.5 * h * e))
                 - (brute_phi(w.basis, sp, d + h * e) - brute_phi(w.basis, sp, d - h * e))) / (6.0 * h)
            s = dV(w) * V * (g * psi).sum(1)
            Fref[C, a] += s.sum()
            sref[a] -= (s[:, None] * d).sum(0) / Omega
    assert np.abs(F - Fref).max() <= 1e-7 * np.abs(Fref).max(), np.abs(F - Fref).max() / np.abs(Fref).max()
    assert np.abs(sigma - sref).max() <= 1e-7 * np.abs(sref).max()
